"""world_size-2 gloo test of the multi-GPU host logic: time-sharding + ordered all-gather sum.

Each rank folds its own contiguous range at its absolute start index (here with the oracle standing
in for the GPU kernels -- this test is about the index arithmetic and the exchange), the bins are
exchanged with ``sharding.allgather_sum`` and must equal the fold of the whole stream."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_range_properties():
    from paper_2501_05993_b200.sharding import shard_range
    for n, world, align in [(1000, 2, 64), (1 << 28, 8, 64), (63, 4, 64), (6400_0001, 3, 4), (0, 2, 16)]:
        edges = [shard_range(n, r, world, align) for r in range(world)]
        assert edges[0][0] == 0 and edges[-1][1] == n
        for (a, b), (c, d) in zip(edges[:-1], edges[1:]):
            assert b == c and a <= b and b % align == 0 or b == n
        sizes = [b - a for a, b in edges]
        assert max(sizes) - min(sizes) <= 2 * align
    with pytest.raises(ValueError):
        shard_range(10, 2, 2, 4)


def _worker(rank, world, port, n, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle as orc
    from paper_2501_05993_b200 import synth
    from paper_2501_05993_b200.sharding import allgather_sum, shard_range
    w = synth.config(2).scaled(n)
    buf = synth.generate(w, "cpu").numpy()
    lo, hi = shard_range(n, rank, world, 64)
    seg = np.ascontiguousarray(buf[lo // 4: (hi + 3) // 4])
    pr, pi = orc.fold_ld(seg, orc.TWO_BIT_OFFSET_BINARY, 1, 0, 0, 1, hi - lo, lo, w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0])
    local = torch.tensor(np.stack([pr.astype(np.float64), pi.astype(np.float64)]))
    total = allgather_sum(local)
    if rank == 0:
        q.put(total.numpy())
    dist.destroy_process_group()


def test_time_sharded_fold_with_gloo_world2(oracle):
    n = 200_004
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    from paper_2501_05993_b200 import synth
    w = synth.config(2).scaled(n)
    buf = synth.generate(w, "cpu").numpy()
    pr, pi = oracle.fold_ld(buf, oracle.TWO_BIT_OFFSET_BINARY, 1, 0, 0, 1, n, 0, w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0])
    assert np.abs(got[0] - pr.astype(np.float64)).max() < 1e-8
    assert np.abs(got[1] - pi.astype(np.float64)).max() < 1e-8
