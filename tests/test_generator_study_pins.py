"""Pins for oracle/generator_study.py (R26).

Expected values come from analysis, not from the emulation itself: in exact arithmetic every
recursion of eq. 2.6 / 2.7 reproduces exp(-j n dphi) (fp64 runs must sit at rounding level); when
2 cos(dphi) rounds to exactly 2.0f the DFR collapses to y[n+1] = 2 y[n] - y[n-1], a straight line
with a closed-form error ("2c_n -> 2.00^-"); the k-shift of PAPER.md:97 removes that
degeneracy; the direct method's error is the rounding of the running float32 phase.
tests/golden/generator_accuracy_survey.txt holds the figures SURVEY.md section 7 measured with an
independent emulation (order-of-magnitude check only).
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import generator_study as gs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "generator_accuracy_survey.txt")


def test_exact_rounding_helper():
    assert gs._round_to(Fraction(1, 3), 24) == float(np.float32(1.0 / 3.0))
    assert gs._round_to(Fraction(-2, 3), 53) == -2.0 / 3.0
    # ties to even at 24 bits: 1 + 2^-24 is a midpoint -> 1.0 ; 1 + 3*2^-24 -> 1 + 2^-22
    assert gs._round_to(1 + Fraction(1, 2 ** 24), 24) == 1.0
    assert gs._round_to(1 + Fraction(3, 2 ** 24), 24) == 1.0 + 2.0 ** -22
    a = gs._Arith(32)
    x, y, z = np.float32(1.0000001), np.float32(3.1415927), np.float32(-3.1415927)
    assert float(a.fma(x, y, z)) == float(np.float32(float(x) * float(y) + float(z)))   # product exact in fp64, sum exact here


@pytest.mark.parametrize("form", [gs.CFO, gs.MCO, gs.DFR, gs.DFR_FMA])
def test_every_recursion_reproduces_the_rotator_in_fp64(form):
    """Sign (exp(-j)), initial values, the Magic Circle's half step: all wrong choices give O(1) errors."""
    err = gs.run(form, 64, 32e6, 10e3 + 3e6, 4096, 4)       # dphi = 0.59 rad: well conditioned
    assert err.max() < 1e-11, err


def test_dfr32_degenerates_when_2cos_rounds_to_two():
    """Config 5: dphi = 2 pi 1234.567/1.024e9 = 7.58e-6 rad, 2 cos(dphi) = 2 - 5.7e-11 -> 2.0f.
    Then cos stays 1 and -sin grows linearly: |error| = |(1 - cos x) + j(sin x - x)|, x = n dphi."""
    f_s, f_off, n = 1024e6, 1234.567, 65536
    dphi = 2 * math.pi * f_off / f_s
    assert np.float32(2 * math.cos(dphi)) == np.float32(2.0)
    err = gs.run(gs.DFR, 32, f_s, f_off, n, 1)[0]
    x = n * dphi
    want = math.hypot(1 - math.cos(x), math.sin(x) - x)
    assert abs(err - want) < 0.02 * want, (err, want)       # 0.123: SURVEY section 7 measured 1.2e-1
    # the k-shift of PAPER.md:97 (k = N_bins/4 -> dphi = pi/2 + ...) removes the degeneracy
    err_k = gs.run(gs.DFR, 32, f_s, f_off + 256 * 1e6, n, 1)[0]
    assert err_k < 1e-4 * err


def test_direct_float32_error_is_the_phase_rounding():
    """K1: phase = float32(n) * float32(dphi); its rounding error grows like n * 2^-24 * dphi... bounded by
    half an ulp of the product plus the relative error of dphi32 times n dphi."""
    f_s, f_off, n = 32e6, 10e3, 20000
    dphi = 2 * math.pi * f_off / f_s
    err = gs.run(gs.DIRECT, 32, f_s, f_off, n, 4)
    rel = abs(float(np.float32(dphi)) - dphi) / dphi
    x = n * dphi
    bound = x * rel + 0.5 * float(np.spacing(np.float32(x))) + 3e-7
    assert err[-1] <= 1.05 * bound and err[-1] > 0.05 * bound, (err, bound)
    assert err[0] < err[-1]                                   # "accuracy declines with n"


def test_orders_of_magnitude_match_the_survey_figures():
    """SURVEY.md section 7, hard part 3 (independent fp32 emulation): max |error| of the phasor."""
    rows = [l.split() for l in open(GOLD).read().splitlines() if l and not l.startswith("#")]
    name = {"CFO": gs.CFO, "MCO": gs.MCO, "DFR": gs.DFR, "DFR_FMA": gs.DFR_FMA}
    for form, prec, f_s, f_rot, n, want in rows:
        got = gs.run(name[form], int(prec), float(f_s), float(f_rot), int(n), 1)[0]
        assert want and float(want) / 4 < got < float(want) * 4, (form, prec, f_rot, n, got, want)
