"""Multi-pass counter-rotation on the device (R27) against oracle/refine.py.

The input carries a comb whose offset differs from the context's nominal f_offset by a known delta; the oracle
side extracts every short integration with oracle/pcal_oracle.c (independent of the GPU path) and runs the same
passes step by step.
"""
import math

import numpy as np
import pytest
import torch

from paper_2501_05993_b200 import binding, synth
from oracle import refine as orefine
from pcal_testlib import oracle_fmt

pytestmark = pytest.mark.gpu


def workload(idx, n, delta):
    w = synth.config(idx).scaled(n)
    true = synth.replace(w, f_offset_hz=[w.f_offset_hz[0] + delta])     # what the data contains
    return w, synth.generate(true, "cuda")


@pytest.mark.parametrize("idx,n_per,M,delta", [(2, 320_000, 6, 12.5), (2, 32_000, 8, -210.0), (1, 64_000, 5, 77.0), (5, 262_144, 4, 300.0)])
def test_residual_rotation_kernel_matches_oracle_estimator(oracle, idx, n_per, M, delta):
    """pcal_residual_rotation on a device series == the oracle's lag-one estimator on the same numbers, and its phase
    is the closed form 2 pi delta T_int (to the noise of the short integrations)."""
    w, dev = workload(idx, n_per * M, delta)
    p = binding.from_workload(w)
    T = torch.empty((M, 1, w.n_bins), dtype=torch.complex128, device="cuda")
    p.extract_series(dev, n_per, M, T)
    got = p.residual_rotation(T, M)[0]
    # (a) the kernel's arithmetic: the oracle's estimator on the very same numbers
    want = orefine.residual_rotation(T.cpu().numpy()[:, 0, :], zero_offset=(w.f_offset_hz[0] == 0.0))
    assert abs(got[0] - want[0]) <= 1e-10
    assert abs(got[1] - want[1]) <= 1e-11 * want[1] and abs(got[2] - want[2]) <= 1e-11 * want[2]
    # (b) end to end, nothing from the GPU on the oracle's side: the oracle's estimator on the ORACLE's series of the
    # same bytes.  Every tone of the GPU series is within 1e-5 of the oracle's, hence arg S within 1e-5 rad.
    host = dev.cpu().numpy().reshape(-1).view(np.uint8)
    bytes_per = n_per * w.bits // 8
    series = np.empty((M, w.n_bins), np.complex128)
    for m in range(M):
        series[m] = oracle.extract(host[m * bytes_per:(m + 1) * bytes_per], oracle_fmt(oracle, w), 1, 0, n_per, m * n_per,
                                   w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0])
    indep = orefine.residual_rotation(series, zero_offset=(w.f_offset_hz[0] == 0.0))
    assert abs(got[0] - indep[0]) <= 1e-5
    assert abs(got[1] - indep[1]) <= 1e-5 * indep[1] and abs(got[2] - indep[2]) <= 1e-5 * indep[2]
    t_int = n_per / w.f_s_hz
    # closed form, to the noise of the short integrations (config 5: comb amplitude 1 under sigma = 20 noise)
    assert abs(got[0] - 2 * math.pi * delta * t_int) < (0.15 if idx == 5 else 0.02)
    p.destroy()


@pytest.mark.parametrize("idx,n_per,M,delta,rot", [(2, 64_000, 8, 41.7, None), (2, 64_000, 8, -133.0, "generator"), (8, 32_000, 6, 95.0, None)])
def test_refine_offset_matches_oracle_passes(oracle, idx, n_per, M, delta, rot):
    """The whole loop: GPU passes vs oracle passes (oracle extraction of the same bytes).  The 1e-5 rad bar on the
    phase maps to 1e-5 / (2 pi T_int) Hz on the refined frequency."""
    w, dev = workload(idx, n_per * M, delta)
    if rot:
        w = synth.replace(w, rotator=rot)
    host = dev.cpu().numpy().reshape(-1).view(np.uint8)
    fmt = oracle_fmt(oracle, w)
    bytes_per = n_per * w.bits // 8

    def series_of(f_rot):
        out = np.empty((M, w.n_bins), np.complex128)
        for m in range(M):
            out[m] = oracle.extract(host[m * bytes_per:(m + 1) * bytes_per], fmt, 1, 0, n_per, m * n_per, w.f_s_hz, w.f_comb_hz, f_rot)
        return out

    f_want, h_want = orefine.refine(series_of, w.f_offset_hz[0], n_per, w.f_s_hz, max_passes=4, tol_rad=1e-4)
    p = binding.from_workload(w)
    f_got, h_got = p.refine_offset(dev, n_per, M, max_passes=4, tol_rad=1e-4)
    t_int = n_per / w.f_s_hz
    assert len(h_got) == len(h_want) >= 2
    for a, b in zip(h_got, h_want):
        assert abs(a[0] - b[0]) <= 1e-5 / (2 * math.pi * t_int) + 1e-6       # rotator frequency of the pass
        assert abs(a[1] - b[1]) <= 1e-5                                        # residual phase shift
        assert abs(a[2] - b[2]) <= 1e-4 * b[2]
    assert abs(f_got - f_want) <= 1e-5 / (2 * math.pi * t_int) + 1e-6
    assert abs(f_got - (w.f_offset_hz[0] + delta)) < 0.02 / (2 * math.pi * t_int)   # close to the truth (noise-limited)
    # the context now carries the refined offset: the long coherent integration follows
    inf = p.info()
    assert inf.n_processed == 0
    p.extract(dev, n_per * M)
    T = p.finalize()
    want = oracle.extract(host, fmt, 1, 0, n_per * M, 0, w.f_s_hz, w.f_comb_hz, f_got)
    rel = np.abs(T[0] - want) / np.abs(want)
    assert rel.max() < 1e-5
    p.destroy()


def test_refine_offset_argument_checks():
    w = synth.config(4).scaled(4096)
    dev = synth.generate(w, "cuda")
    p = binding.from_workload(w)
    with pytest.raises(binding.PcalError) as e:
        p.refine_offset(dev, 1024, 4)
    assert e.value.code == -4            # multi-channel: unsupported
    p.destroy()
    w = synth.config(2).scaled(1 << 16)
    dev = synth.generate(w, "cuda")
    p = binding.from_workload(w)
    with pytest.raises(binding.PcalError) as e:
        p.refine_offset(dev, 1 << 15, 1)
    assert e.value.code == -1            # fewer than two periods
    p.destroy()
