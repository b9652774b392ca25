"""world_size-2 gloo test of the multi-GPU host logic: time-sharding + ordered all-gather sum.

Each rank folds its own contiguous range at its absolute start index (here with the oracle standing
in for the GPU kernels -- this test is about the index arithmetic and the exchange), the bins are
exchanged by ``sharding.ShardedIntegrator`` / ``sharding.series_sharded`` -- the code path bench.py --gpus N runs -- and must
equal the extraction of the whole stream."""
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


class OracleContext:
    """Stand-in for ``binding.Pcal`` where there is no GPU: the seven calls ``sharding`` makes, answered by the oracle
    on CPU tensors (this test is about the index arithmetic and the exchange; the sum that pcal_set_folded_sum_dev does
    on the device is a rank-order loop here)."""

    def __init__(self, orc, w):
        self.orc, self.w, self.start = orc, w, 0
        self.P = np.zeros((w.n_bins,), np.complex128)

    def reset(self):
        self.P[:] = 0
        self.start = 0

    def set_start_index(self, n):
        self.start = n

    def extract(self, samples, n):
        w = self.w
        pr, pi = self.orc.fold_ld(samples.numpy(), self.orc.TWO_BIT_OFFSET_BINARY, 1, 0, 0, 1, n, self.start,
                                  w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0])
        self.P += pr.astype(np.float64) + 1j * pi.astype(np.float64)
        self.start += n

    def get_folded_dev(self, t):
        t.copy_(torch.from_numpy(self.P.view(np.float64).copy()))

    def set_folded_sum_dev(self, parts, n_parts):
        parts = parts.numpy().reshape(n_parts, -1)
        acc = np.zeros_like(parts[0])
        for r in range(n_parts):
            acc = acc + parts[r]
        self.P = acc.view(np.complex128).copy()

    def finalize_async(self, out):
        out.copy_(torch.from_numpy(self.orc.dft(self.P.real.astype(np.longdouble), self.P.imag.astype(np.longdouble))))

    def finalize_series_sum_dev(self, parts, n_parts, m, out_folded, out_tones):
        parts = parts.numpy().reshape(n_parts, m, -1)
        for k in range(m):
            acc = np.zeros_like(parts[0, k])
            for r in range(n_parts):
                acc = acc + parts[r, k]
            z = acc.view(np.complex128)
            out_folded[k, 0].copy_(torch.from_numpy(z.copy()))
            out_tones[k, 0].copy_(torch.from_numpy(self.orc.dft(z.real.astype(np.longdouble), z.imag.astype(np.longdouble))))


def _worker(rank, world, port, n, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle as orc
    orc.build()
    from paper_2501_05993_b200 import synth
    from paper_2501_05993_b200.sharding import ShardedIntegrator, series_sharded, shard_range
    w = synth.config(2).scaled(n)
    buf = synth.generate(w, "cpu")
    lo, hi = shard_range(n, rank, world, 64)
    seg = buf[lo // 4: (hi + 3) // 4].contiguous()
    # (a) three periods through two lanes: the product's own code path (bench.py --gpus N runs exactly this class)
    s = ShardedIntegrator([OracleContext(orc, w), OracleContext(orc, w)], 1, w.n_bins, world, "cpu")
    outs = [torch.zeros(w.n_bins, dtype=torch.complex128) for _ in range(3)]
    for o in outs:
        s.submit(seg, hi - lo, lo, o)
    s.drain()
    # (b) a series of two periods (the two halves of the stream), one exchange for both
    half = n // 2 - (n // 2) % 128
    shards, starts = [], []
    for k in range(2):
        a, b = shard_range(half, rank, world, 64)
        shards.append(buf[(k * half + a) // 4: (k * half + b + 3) // 4].contiguous())
        starts.append(k * half + a)
    pf = torch.zeros((2, 1, w.n_bins), dtype=torch.complex128)
    pt = torch.zeros((2, 1, w.n_bins), dtype=torch.complex128)
    a, b = shard_range(half, rank, world, 64)
    series_sharded(OracleContext(orc, w), shards, b - a, starts, 1, w.n_bins, world, "cpu", pf, pt)
    if rank == 0:
        q.put(([o.numpy() for o in outs], pf.numpy(), pt.numpy(), half))
    dist.destroy_process_group()


def test_time_sharded_integrations_with_gloo_world2(oracle):
    n = 200_064
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, q)) for r in range(2)]
    for p in procs:
        p.start()
    outs, pf, pt, half = q.get(timeout=180)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    from paper_2501_05993_b200 import synth
    w = synth.config(2).scaled(n)
    buf = synth.generate(w, "cpu").numpy()
    pr, pi = oracle.fold_ld(buf, oracle.TWO_BIT_OFFSET_BINARY, 1, 0, 0, 1, n, 0, w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0])
    want = oracle.dft(pr, pi)
    for o in outs:
        assert np.abs(o - want).max() < 1e-9 * np.abs(want).max()
    for k in range(2):
        seg = buf[k * half // 4: (k + 1) * half // 4]
        pr, pi = oracle.fold_ld(seg, oracle.TWO_BIT_OFFSET_BINARY, 1, 0, 0, 1, half, k * half, w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0])
        assert np.abs(pf[k, 0] - (pr.astype(np.float64) + 1j * pi.astype(np.float64))).max() < 1e-8
        wt = oracle.dft(pr, pi)
        assert np.abs(pt[k, 0] - wt).max() < 1e-9 * np.abs(wt).max()
