"""GPU parity of pcal_analyze against oracle/analysis.py on the same seeded bytes.

Oracle side: C oracle fold (long double) -> DFT -> plain fp64 analysis.  CUDA side: everything
through the C ABI.  Integer outputs (arg-max bin) must be equal; delays, slopes and the corrected
band-pass agree to tolerances that follow from north_star's 1e-5 per tone.
"""
import math

import numpy as np
import pytest
import torch

from oracle import analysis as ana
from paper_2501_05993_b200 import binding, synth
from pcal_testlib import assert_close, oracle_folded

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("idx,n,rot", [(1, 1_300_001, None), (2, 2_000_004, None), (3, 2_600_036, None),
                                       (3, 1_300_004, "generator"), (4, 200_003, None), (5, 1_300_003, None)])
def test_analyze_matches_oracle(oracle, idx, n, rot):
    w = synth.config(idx).scaled(n)
    if rot:
        w = synth.replace(w, rotator=rot)
    dev = synth.generate(w, "cuda")
    host = dev.cpu().numpy()
    p = binding.from_workload(w)
    p.extract(dev, n)
    summ, B = p.analyze()
    for c in range(0, w.n_channels, 5):
        pr, pi = oracle_folded(oracle, w, host, c)
        P = pr.astype(np.float64) + 1j * pi.astype(np.float64)
        T = oracle.dft(pr, pi)
        want, wantB = ana.analyze(P, T, w.f_s_hz, w.f_comb_hz, w.f_offset_hz[c])
        got = summ[c]
        assert got[0] == want[0], (idx, c, got[0], want[0])                 # arg-max bin: exact
        # the two analyses start from bins/tones that agree to REL_TOL = 1e-5 (float32 / generator paths;
        # ~1e-13 on the integer paths): powers to 2e-5, the vertex to 1e-4 bin, every phase to 1e-5 rad
        assert abs(got[1] - want[1]) < 1e-4
        assert abs(got[2] - want[2]) < 1e-4 / w.f_s_hz
        assert abs(got[3] - want[3]) <= 2e-5 * want[3] and abs(got[4] - want[4]) <= 2e-5 * want[4]
        assert abs(got[5] - want[5]) < 1e-5 / (2 * math.pi * w.f_comb_hz)
        assert abs(got[6] - want[6]) < 1e-5 and abs(got[7] - want[7]) < 1e-5
        K = w.n_bins // 2
        first = 0 if w.f_offset_hz[c] else 1
        assert_close(B[c][first:K], wantB[first:K], f"cfg{idx} ch{c} corrected band-pass")
    # analysis does not disturb the accumulators: finalize still gives the same spectrum
    T1 = p.finalize()
    p.analyze(bandpass=False)
    assert np.array_equal(T1, p.finalize())
    p.destroy()


def test_analyze_recovers_the_synthetic_cable_delay():
    """End to end on noisy 2-bit data: the phase-slope delay lands on config 2's t_d = 5 ns."""
    w = synth.config(2).scaled(1 << 24)
    dev = synth.generate(w, "cuda")
    p = binding.from_workload(w)
    p.extract(dev, w.n_samples)
    summ, _ = p.analyze(bandpass=False)
    assert abs(summ[0][5] - 5e-9) < 0.5e-9          # 16.7 M samples of sigma = 1 noise, 16 tones of 0.05
    pos = (summ[0][0] + summ[0][1]) % w.n_bins       # pulse sits at -t_d f_s = -0.16 samples (mod N_bins)
    assert min(pos, w.n_bins - pos) < 0.5
    p.destroy()
