"""GPU parity of pcal_generator_study against oracle/generator_study.py.

fp32/fp64 recursions are sequences of single correctly rounded operations on both sides, so the
generated states are bit-identical and the recorded errors differ only through the fp64 evaluation
of the exact phasor (~1e-16); the direct method goes through cosf/sinf of the two libraries (1-2 ulp
of float32).  Then the paper's qualitative claims at full length.
"""
import numpy as np
import pytest

from oracle import generator_study as gs
from paper_2501_05993_b200 import binding

pytestmark = pytest.mark.gpu

CASES = [(form, prec, f_s, f_rot)
         for (f_s, f_rot) in [(1024e6, 1234.567), (32e6, 10e3), (1024e6, 256e6 + 1234.567), (16e6, 10e3 + 3e6)]
         for form in (gs.CFO, gs.MCO, gs.DFR, gs.DFR_FMA) for prec in (32, 64)] + \
        [(gs.DIRECT, 32, 32e6, 10e3), (gs.DIRECT, 32, 1024e6, 1234.567)]


def test_errors_match_the_step_by_step_oracle():
    n, n_chk = 20000, 5
    got = binding.generator_study(CASES, n, n_chk)
    for row, (form, prec, f_s, f_rot) in zip(got, CASES):
        want = gs.run(form, prec, f_s, f_rot, n, n_chk)
        tol = 5e-7 if form == gs.DIRECT else 1e-12
        assert np.abs(row - want).max() <= tol + 1e-9 * want.max(), (form, prec, f_s, f_rot, row, want)


def test_paper_claims_over_a_million_cycles():
    """low dphi distorts the fp32 DFR; :97 a k-shift reduces the error significantly;
    :95 double precision reduces it; :142/505 the direct method declines with n."""
    n = 1 << 20
    f_s, f_off = 1024e6, 1234.567
    cases = [(gs.DFR, 32, f_s, f_off), (gs.DFR, 32, f_s, f_off + 256e6), (gs.DFR, 64, f_s, f_off),
             (gs.CFO, 32, f_s, f_off), (gs.MCO, 32, f_s, f_off), (gs.DIRECT, 32, 32e6, 10e3)]
    e = binding.generator_study(cases, n, 8)
    dfr32, dfr32_k, dfr64, cfo32, mco32, direct = e
    assert dfr32[-1] > 0.5                       # degenerate: 2cos(dphi) == 2.0f
    assert dfr32_k[-1] < 1e-3 * dfr32[-1]
    assert dfr64[-1] < 1e-3 * dfr32[-1]
    assert mco32[-1] < 1e-3 and cfo32[-1] < 1e-2
    assert direct[-1] > 5 * direct[0]            # accuracy declines with n (linear growth over 8 intervals)


def test_argument_checks():
    with pytest.raises(binding.PcalError):
        binding.generator_study([(7, 32, 32e6, 10e3)], 10, 1)
    with pytest.raises(binding.PcalError):
        binding.generator_study([(gs.CFO, 16, 32e6, 10e3)], 10, 1)
