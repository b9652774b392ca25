"""Time-sharding of an integration across ranks (PAPER.md:13, 527:
"multi-core processing" -- segment the stream, add the partial bins).

eq. 2.2 is a running sum over the sample index, so a stream can be cut into contiguous time ranges,
each rank folding its own range *at its absolute start index* (bin index and rotator phase then line
up), followed by ONE exchange: the sum over ranks of the n_channels x N_bins complex bins
(<= 16 KiB).  For a deterministic fp64 result the exchange is an all-gather followed by a sum in
rank order on every rank (not an all-reduce, whose order is not fixed); the sum itself runs in the
library (pcal_set_folded_sum_dev / pcal_finalize_series_sum_dev), never in torch.

This module is host logic only: index arithmetic and torch.distributed plumbing around a *context*
-- ``binding.Pcal`` on a GPU (NCCL), or any object with the same seven methods (the gloo CPU test
passes one backed by the oracle).  It contains none of the extraction arithmetic.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Tuple

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


def _all_gather(gathered: torch.Tensor, local: torch.Tensor, group=None):
    """Default exchange: one all-gather into a flat [world * len(local)] tensor, asynchronous."""
    return dist.all_gather_into_tensor(gathered, local, group=group, async_op=True)


class ShardedIntegrator:
    """Integration periods whose samples are spread over ``world`` ranks in time.

    ``submit`` enqueues one period on this rank -- reset, fold the local shard at its absolute start
    index, hand the bins to the all-gather -- and returns without waiting; the period is *completed*
    (rank-order sum, DFT, tones into ``out``) when its lane comes round again or on ``drain``.  With
    two lanes the all-gather of period k is in flight while period k+1 is folded and period k-1 is
    finished.  ``contexts``: one context per lane, all created with the same parameters.
    """

    def __init__(self, contexts: List, n_channels: int, n_bins: int, world: int, device,
                 gather: Optional[Callable] = None, group=None):
        self.world, self.group = world, group
        self.gather = gather or (lambda gathered, local: _all_gather(gathered, local, group))
        n = n_channels * n_bins * 2
        self.lanes = [{"ctx": c, "work": None, "out": None,
                       "local": torch.empty(n, dtype=torch.float64, device=device),
                       "gathered": torch.empty(world * n, dtype=torch.float64, device=device)} for c in contexts]
        self.count = 0

    def _complete(self, lane):
        if lane["work"] is not None:
            lane["work"].wait()                            # the current stream waits for the all-gather
            lane["ctx"].set_folded_sum_dev(lane["gathered"], self.world)
            lane["ctx"].finalize_async(lane["out"])
            lane["work"] = None

    def submit(self, dev_samples, n_local: int, start_index: int, out):
        lane = self.lanes[self.count % len(self.lanes)]
        self._complete(lane)                               # this lane's previous period, if still open
        ctx = lane["ctx"]
        ctx.reset()
        ctx.set_start_index(start_index)
        ctx.extract(dev_samples, n_local)
        ctx.get_folded_dev(lane["local"])
        lane["out"] = out
        lane["work"] = self.gather(lane["gathered"], lane["local"])
        self.count += 1
        if len(self.lanes) > 1:
            self._complete(self.lanes[self.count % len(self.lanes)])   # finish the other lane under this all-gather

    def drain(self):
        for lane in self.lanes:
            self._complete(lane)


def integrate_sharded(ctx, dev_samples, n_local: int, start_index: int, out, n_channels: int, n_bins: int, world: int,
                      device, gather: Optional[Callable] = None, group=None):
    """One period, one lane: fold the local shard, exchange, finish.  ``out`` receives the tones of the
    WHOLE period on every rank (asynchronously: the caller synchronises its stream)."""
    s = ShardedIntegrator([ctx], n_channels, n_bins, world, device, gather, group)
    s.submit(dev_samples, n_local, start_index, out)
    s.drain()


def series_sharded(ctx, period_shards, n_local: int, period_starts, n_channels: int, n_bins: int, world: int, device,
                   out_folded: torch.Tensor, out_tones: torch.Tensor, gather: Optional[Callable] = None, group=None):
    """A time series of M periods with ONE exchange: ``period_shards[k]`` = this rank's samples of period k,
    ``period_starts[k]`` = their absolute start index.  Every period is folded locally, the M sets of bins
    travel in one all-gather, and the library adds them in rank order and takes the M DFTs.
    ``out_folded`` / ``out_tones``: device tensors [M, n_channels, n_bins] complex128."""
    m = len(period_shards)
    n = n_channels * n_bins * 2
    local = torch.empty(m * n, dtype=torch.float64, device=device)
    gathered = torch.empty(world * m * n, dtype=torch.float64, device=device)
    for k in range(m):
        ctx.reset()
        ctx.set_start_index(period_starts[k])
        ctx.extract(period_shards[k], n_local)
        ctx.get_folded_dev(local[k * n:(k + 1) * n])
    work = (gather or (lambda g, l: _all_gather(g, l, group)))(gathered, local)
    work.wait()
    ctx.finalize_series_sum_dev(gathered, world, m, out_folded, out_tones)
