"""pcal_extract_series: a time series of integrations in one call.

Period k must equal the oracle's fold + DFT of the samples [k, k+1)*n_per_period with the absolute
sample index running on (n_abs0 = k*n_per_period): the rotator phase is continuous across periods.
"""
import numpy as np
import pytest
import torch

from paper_2501_05993_b200 import binding, synth
from pcal_testlib import assert_close, oracle_fmt

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("idx,n_per,n_periods,rot", [(2, 320_064, 5, None), (4, 40_004, 4, None), (5, 262_160, 3, None),
                                                     (1, 100_004, 3, None), (3, 512_000, 3, "generator"), (4, 40_064, 3, "generator")])
def test_series_matches_per_period_oracle(oracle, idx, n_per, n_periods, rot):
    w = synth.config(idx).scaled(n_per * n_periods)
    if rot:
        w = synth.replace(w, rotator=rot)
    dev = synth.generate(w, "cuda")
    host = dev.cpu().numpy().reshape(-1).view(np.uint8)
    p = binding.from_workload(w)
    T = torch.empty((n_periods, w.n_channels, w.n_bins), dtype=torch.complex128, device="cuda")
    P = torch.empty_like(T)
    p.extract_series(dev, n_per, n_periods, T, P)
    torch.cuda.synchronize()
    assert p.info().n_processed == n_per * n_periods
    T, P = T.cpu().numpy(), P.cpu().numpy()
    fmt = oracle_fmt(oracle, w)
    bytes_per = n_per * w.bits * w.n_channels // 8
    for k in range(n_periods):
        seg = host[k * bytes_per:(k + 1) * bytes_per]
        for c in range(0, w.n_channels, 7):
            pr, pi = oracle.fold_ld(seg, fmt, w.n_channels, c, 0, 1, n_per, k * n_per,
                                    w.f_s_hz, w.f_comb_hz, w.f_offset_hz[c], tabulated=True, threads=1)
            assert_close(P[k, c], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"cfg{idx} period {k} ch{c} folded", max_small=1)
            assert_close(T[k, c], oracle.dft(pr, pi), f"cfg{idx} period {k} ch{c} tones", max_small=1)
    # the context is left with the last period: finalize repeats it
    Tl = p.finalize()                                # (the DFT kernel and the fold kernel's own DFT sum in different orders)
    assert np.abs(Tl - T[-1]).max() <= 1e-12 * np.abs(Tl).max()
    p.destroy()


def test_series_alignment_and_empty():
    w = synth.config(2).scaled(1 << 16)
    dev = synth.generate(w, "cuda")
    p = binding.from_workload(w)
    T = torch.empty((2, 1, w.n_bins), dtype=torch.complex128, device="cuda")
    with pytest.raises(binding.PcalError) as e:
        p.extract_series(dev, 100, 2, T)            # 200 bits per period: not a multiple of 128
    assert e.value.code == -2
    p.extract_series(dev, 0, 2, T)                   # no-op
    p.extract_series(dev, 1 << 15, 0, T)             # no-op
    assert p.info().n_processed == 0
    p.destroy()
