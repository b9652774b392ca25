"""TEST INFRASTRUCTURE, NOT THE PRODUCT -- plain fp64 restatement of the multi-pass counter-rotation.

SURVEY.md section 8(f)4 / PAPER.md:49: "Picosecond accuracy can be reached with long integration times, or
alternatively, short integration times combined with multiple passes over the x[n] input data, iteratively
counter-rotating the input data using the residual phase shift detected in the previous pass."  The paper
gives one sentence and no formula; reading R27 fixes it:

  * a PASS is a time series of M short integrations of N_int samples each over the SAME stored input
    (PAPER.md:126, 138), extracted with the rotator of eq. 2.3 at the current frequency f_rot;
  * the RESIDUAL PHASE SHIFT of a pass is the common phase advance of the tone phasors from one short
    integration to the next.  If the comb really sits at i f_comb + f_true, eq. 2.3 with f_rot leaves every
    tone turning at delta = f_true - f_rot, so T_m[i] = T_0[i] e^{+j 2 pi delta T_int m}, T_int = N_int/f_s,
    and the lag-one product sum   S = sum_{m=0}^{M-2} sum_{i in band} T_{m+1}[i] conj(T_m[i])
    has  arg S = 2 pi delta T_int  (unambiguous for |delta| < 1/(2 T_int): hence SHORT integrations);
  * the next pass COUNTER-ROTATES by that shift: f_rot <- f_rot + arg S / (2 pi T_int), snapped to the
    1 micro-hertz grid (R16);  passes repeat until |arg S| <= tol or max_passes is reached;
  * in band = tones 1 .. N_bins/2 - 1 when f_rot starts at 0, else 0 .. N_bins/2 - 1 (R4, R5).

Everything is written step by step with Python/numpy fp64 scalars so that it can be checked against the
text by eye.  Shares no code with paper_2501_05993_b200/.  Pins: tests/test_refine_pins.py (closed form of
the lag-one product for a pure rotation, invariance to a common amplitude/phase, end-to-end recovery of a
known offset from the oracle's own extraction of a noise-free comb, second pass ~ 0).
"""
from __future__ import annotations

import math

import numpy as np

N_RESIDUAL = 3  # dtheta_rad, |S|, sum of |T_{m+1}||T_m| (|S| / this = coherence in [0, 1])


def in_band(n_bins: int, zero_offset: bool):
    """Tone indices that carry comb power (R4, R5)."""
    return range(1 if zero_offset else 0, n_bins // 2)


def residual_rotation(T: np.ndarray, zero_offset: bool):
    """T: complex [M, N_bins] tone spectra of M consecutive short integrations (one channel).
    Returns (arg S, |S|, sum |T_{m+1}[i]| |T_m[i]|); S as in the module text, summed m-major, i-minor."""
    M, N = T.shape
    s_re, s_im, norm = 0.0, 0.0, 0.0
    for m in range(M - 1):
        for i in in_band(N, zero_offset):
            a, b = complex(T[m + 1, i]), complex(T[m, i])
            # a * conj(b)
            s_re += a.real * b.real + a.imag * b.imag
            s_im += a.imag * b.real - a.real * b.imag
            norm += math.sqrt(a.real * a.real + a.imag * a.imag) * math.sqrt(b.real * b.real + b.imag * b.imag)
    return math.atan2(s_im, s_re), math.hypot(s_re, s_im), norm


def next_rotator_hz(f_rot_hz: float, dtheta_rad: float, n_int: int, f_s_hz: float) -> float:
    """Counter-rotation of the next pass: f_rot + dtheta / (2 pi T_int), on the 1 micro-hertz grid."""
    t_int = n_int / f_s_hz
    return round((f_rot_hz + dtheta_rad / (2.0 * math.pi * t_int)) * 1e6) / 1e6


def refine(series_of, f_rot0_hz: float, n_int: int, f_s_hz: float, max_passes: int, tol_rad: float):
    """series_of(f_rot_hz) -> complex [M, N_bins] (one pass over the stored input at that rotator frequency).
    Returns (final f_rot, history [(f_rot used, dtheta, |S|, norm), ...])."""
    f = f_rot0_hz
    hist = []
    for _ in range(max_passes):
        T = series_of(f)
        dth, mag, norm = residual_rotation(T, zero_offset=(f_rot0_hz == 0.0))
        hist.append((f, dth, mag, norm))
        if abs(dth) <= tol_rad:
            break
        f = next_rotator_hz(f, dth, n_int, f_s_hz)
    return f, hist
