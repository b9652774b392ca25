"""Time-sharding of one integration across ranks.

eq. 2.2 is a running sum over the sample index, so a stream can be cut into contiguous time ranges,
each rank folding its own range *at its absolute start index* (bin index and rotator phase then line
up), followed by ONE exchange: the sum over ranks of the n_channels x N_bins complex bins
(<= 16 KiB).  For a deterministic fp64 result the exchange is an all-gather followed by a sum in
rank order on every rank (not an all-reduce, whose order is not fixed).

This module is host logic only (index arithmetic + torch.distributed plumbing); it contains none of
the extraction arithmetic and works with the gloo backend on CPU tensors and with NCCL on CUDA
tensors alike.
"""
from __future__ import annotations

from typing import Tuple

import torch
import torch.distributed as dist


def shard_range(n_samples: int, rank: int, world: int, align: int) -> Tuple[int, int]:
    """Contiguous [start, stop) of rank ``rank``; every boundary except the last is a multiple of
    ``align`` samples (align = samples per 16 bytes so each shard's pointer stays 16-byte aligned)."""
    if world < 1 or not (0 <= rank < world) or align < 1:
        raise ValueError("bad shard arguments")
    units = -(-n_samples // align)
    per, extra = divmod(units, world)
    lo_u = rank * per + min(rank, extra)
    hi_u = lo_u + per + (1 if rank < extra else 0)
    return min(lo_u * align, n_samples), min(hi_u * align, n_samples)


def allgather_sum(local_bins: torch.Tensor, group=None) -> torch.Tensor:
    """Sum of every rank's bins, added in rank order (bit-identical on all ranks)."""
    world = dist.get_world_size(group)
    parts = [torch.empty_like(local_bins) for _ in range(world)]
    dist.all_gather(parts, local_bins.contiguous(), group=group)
    total = torch.zeros_like(local_bins)
    for p in parts:
        total += p
    return total
