"""Pins of oracle/refine.py (multi-pass counter-rotation; R27) -- CPU only.

What fixes the estimator independently of itself: the closed form of a pure rotation (eq. 2.3 with a
wrong f_rot leaves every tone turning at f_true - f_rot), its invariance to whatever is common to all
periods, and an end-to-end recovery of a known offset from the oracle's OWN extraction (oracle/pcal_oracle.c)
of a noise-free comb per eq. 2.1.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import refine


def rotating_series(M, N, delta_hz, t_int, seed=0):
    """T_m[i] = A_i e^{j psi_i} e^{j 2 pi delta T_int m} typed directly from the text (not from residual_rotation)."""
    rng = np.random.default_rng(seed)
    A = rng.uniform(0.5, 2.0, N) * np.exp(1j * rng.uniform(-np.pi, np.pi, N))
    return np.array([A * np.exp(2j * np.pi * delta_hz * t_int * m) for m in range(M)])


@pytest.mark.parametrize("delta", [0.0, 1.0, -37.5, 123.456, -499.0])
def test_lag_one_phase_is_two_pi_delta_t(delta):
    t_int = 1e-3                                   # |delta| < 1/(2 T_int) = 500 Hz
    T = rotating_series(6, 32, delta, t_int)
    dth, mag, norm = refine.residual_rotation(T, zero_offset=False)
    assert abs(dth - 2 * math.pi * delta * t_int) < 1e-12
    assert abs(mag / norm - 1.0) < 1e-12           # fully coherent
    f1 = refine.next_rotator_hz(10e3, dth, 32000, 32e6)
    assert abs(f1 - (10e3 + delta)) <= 1e-6        # 1 micro-hertz grid


def test_sign_convention_and_aliasing():
    t_int = 1e-3
    T = rotating_series(4, 16, +100.0, t_int)
    assert refine.residual_rotation(T, False)[0] > 0          # tones advancing <=> f_true above f_rot
    assert refine.residual_rotation(np.conj(T), False)[0] < 0
    # beyond the unambiguous range the estimate wraps by 1/T_int
    T = rotating_series(4, 16, 700.0, t_int)
    dth = refine.residual_rotation(T, False)[0]
    assert abs(dth - 2 * math.pi * (700.0 - 1000.0) * t_int) < 1e-12


def test_invariant_to_common_factor_and_band_selection():
    t_int, delta = 2e-3, 40.0
    T = rotating_series(5, 32, delta, t_int, seed=3)
    a = refine.residual_rotation(T, False)
    b = refine.residual_rotation(T * (3.7 * np.exp(1j * 1.234)), False)
    assert abs(a[0] - b[0]) < 1e-13 and abs(b[1] / a[1] - 3.7 ** 2) < 1e-12
    # upper half of the bins (mirror band, R4) and tone 0 at zero offset (R5) are not used
    T2 = T.copy(); T2[:, 16:] = 1e9 * np.exp(1j * np.arange(16))
    assert abs(refine.residual_rotation(T2, False)[0] - a[0]) < 1e-13
    T3 = T.copy(); T3[:, 0] = 1e9
    assert abs(refine.residual_rotation(T3, True)[0] - refine.residual_rotation(T, True)[0]) < 1e-13
    assert list(refine.in_band(32, True)) == list(range(1, 16)) and list(refine.in_band(32, False)) == list(range(16))


def test_end_to_end_recovers_a_known_offset_from_the_oracle_extraction():
    """Noise-free comb per eq. 2.1 at f_true = 10 kHz + 37.5 Hz, extracted by the C oracle at f_rot = 10 kHz in
    8 periods of 1 ms: pass 1 finds +37.5 Hz (to the leakage between tones), pass 2 finds ~0."""
    f_s, f_comb, f_nom, delta = 32e6, 1e6, 10e3, 37.5
    n_int, M, N = 32000, 8, 32
    n = np.arange(n_int * M, dtype=np.float64)
    td = 5e-9
    x = np.zeros(n.size)
    for i in range(N // 2):
        f_i = i * f_comb + f_nom + delta
        x += np.sin(2 * np.pi * f_i * (n / f_s) + 2 * np.pi * f_i * td)
    x = x.astype(np.float32)

    def series_of(f_rot):
        out = np.empty((M, N), np.complex128)
        for m in range(M):
            out[m] = oracle.extract(x[m * n_int:(m + 1) * n_int], oracle.F32, 1, 0, n_int, m * n_int, f_s, f_comb, f_rot)
        return out

    f, hist = refine.refine(series_of, f_nom, n_int, f_s, max_passes=4, tol_rad=1e-7)
    assert abs(hist[0][1] - 2 * math.pi * delta * n_int / f_s) < 1e-5    # leakage between tones, float32 samples
    assert abs(f - (f_nom + delta)) < 1e-3
    assert len(hist) >= 2 and abs(hist[1][1]) < 1e-5
    assert hist[-1][2] / hist[-1][3] > 0.999999
