"""TEST INFRASTRUCTURE, NOT THE PRODUCT -- plain fp64 restatement of the paper's PCal data analysis.

SURVEY.md section 8(f)1 / PAPER.md:49, 132-136: from the folded period P (eq. 2.2) and its DFT
 the analysis reads
  * the pulse (group) delay "as the position of the maximum power", refined across
    "the neighboring bins around the largest component"; bin i <-> delay i/f_s;
  * the group-delay corrected band-pass profile (Fig. 5);
  * the cable delay t_d of eq. 2.1 from the phase slope across the tones: phi_i =
    (i w_comb + w_offset) t_d f_s, i.e. phase is linear in the tone index.
The paper gives no formulas for the refinement ("for example a hyperbolic estimate") nor for the
fit; readings R23-R25 fix them: three-point vertex on the power envelope, sequential
phase unwrapping, unweighted least squares with a free intercept.

Everything is written step by step with Python/numpy fp64 scalars so that it can be checked
against the text by eye.  Shares no code with paper_2501_05993_b200/.
Pins: tests/test_analysis_pins.py (exact parabola, impulse, closed form of eq. 2.1, steep ramps).
"""
from __future__ import annotations

import math

import numpy as np

N_SUMMARY = 8  # peak_bin, peak_frac, pulse_delay_s, peak_power, total_power, slope_delay_s, intercept_rad, fit_rms_rad


def pulse_peak(P: np.ndarray):
    """(b*, delta, power[b*], sum power): largest |P[b]|^2 (first one on ties) and the vertex of the
    parabola through it and its two cyclic neighbours, delta in (-1/2, 1/2)."""
    N = len(P)
    w = [P[b].real * P[b].real + P[b].imag * P[b].imag for b in range(N)]
    b_star = 0
    for b in range(1, N):
        if w[b] > w[b_star]:
            b_star = b
    ym, y0, yp = w[(b_star - 1) % N], w[b_star], w[(b_star + 1) % N]
    denom = ym - 2.0 * y0 + yp
    delta = 0.5 * (ym - yp) / denom if denom != 0.0 else 0.0
    total = 0.0
    for b in range(N):
        total += w[b]
    return b_star, delta, y0, total


def bandpass_corrected(T: np.ndarray, b_star: int, delta: float) -> np.ndarray:
    """B[i] = T[i] exp(+j 2 pi i (b* + delta)/N): the linear phase of a pulse sitting at b* + delta
    removed (a pulse at position m has DFT exp(-j 2 pi i m/N)).  i*b* is reduced mod N in integers."""
    N = len(T)
    B = np.empty(N, np.complex128)
    for i in range(N):
        ang = 2.0 * math.pi * (((i * b_star) % N) / N + i * delta / N)
        B[i] = T[i] * complex(math.cos(ang), math.sin(ang))
    return B


def phase_slope(T: np.ndarray, first_tone: int, n_tones: int):
    """Unwrapped tone phases theta_i = arg T[i] + pi/2 (eq. 2.1 uses sines, R2) for
    i = first_tone .. n_tones-1, then the least-squares line theta ~ a + s*i.
    Returns (s, a, rms residual).  A comb fixes the delay only modulo 1/f_comb: wrapping every
    step into [-pi, pi) selects the branch |t_d| < 1/(2 f_comb)."""
    idx = list(range(first_tone, n_tones))
    theta = []
    prev = None
    for i in idx:
        th = math.atan2(T[i].imag, T[i].real) + 0.5 * math.pi
        if prev is not None:
            d = th - prev
            d -= 2.0 * math.pi * math.floor(d / (2.0 * math.pi) + 0.5)   # wrap the step into [-pi, pi)
            th = prev + d
        theta.append(th)
        prev = th
    n = len(idx)
    sx = sy = sxx = sxy = 0.0
    for i, th in zip(idx, theta):
        sx += i; sy += th; sxx += i * i; sxy += i * th
    det = n * sxx - sx * sx
    s = (n * sxy - sx * sy) / det if det != 0.0 else 0.0
    a = (sy - s * sx) / n
    rss = 0.0
    for i, th in zip(idx, theta):
        r = th - (a + s * i)
        rss += r * r
    return s, a, math.sqrt(rss / n)


def analyze(P: np.ndarray, T: np.ndarray, f_s_hz: float, f_comb_hz: float, f_offset_hz: float):
    """One channel: (summary[N_SUMMARY], corrected band-pass B[N_bins])."""
    N = len(P)
    b_star, delta, peak, total = pulse_peak(P)
    first = 0 if f_offset_hz != 0.0 else 1          # tone 0 is sin(0) = 0 at f_offset = 0 (R5)
    s, a, rms = phase_slope(T, first, N // 2)
    summary = np.array([float(b_star), delta, (b_star + delta) / f_s_hz, peak, total,
                        s / (2.0 * math.pi * f_comb_hz), a, rms], np.float64)
    return summary, bandpass_corrected(T, b_star, delta)
