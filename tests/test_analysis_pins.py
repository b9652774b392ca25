"""Pins for oracle/analysis.py (PCal data analysis; R23-R25).

Expected values come from closed forms, never from re-typing the oracle's own formula:
an exactly parabolic power profile has a known vertex; an impulse at bin m has DFT
exp(-j 2 pi i m / N); eq. 2.1 with s[n] = 0 fixes every tone phase (phi_i - pi/2) and the pulse
shape (a Dirichlet kernel centred at -t_d f_s); a steep phase ramp must survive unwrapping.
"""
import cmath
import math

import numpy as np
import pytest

from oracle import analysis as ana


def test_three_point_vertex_is_exact_on_a_parabola():
    N, b0, true_delta = 16, 5, 0.3125
    w = np.array([max(0.0, 100.0 - 7.0 * (b - (b0 + true_delta)) ** 2) for b in range(N)])
    P = np.sqrt(w).astype(np.complex128) * cmath.exp(0.7j)          # power = w exactly enough
    b_star, delta, peak, total = ana.pulse_peak(P)
    assert b_star == b0
    assert abs(delta - true_delta) < 1e-12
    assert abs(peak - w[b0]) < 1e-10 and abs(total - w.sum()) < 1e-9


def test_peak_wraps_cyclically_and_ties_take_the_first_bin():
    P = np.zeros(8, np.complex128)
    P[0], P[7], P[1] = 3.0, 2.0, 1.0            # neighbours of bin 0 are bins 7 and 1
    b_star, delta, _, _ = ana.pulse_peak(P)
    assert b_star == 0
    ym, y0, yp = 4.0, 9.0, 1.0
    assert abs(delta - 0.5 * (ym - yp) / (ym - 2 * y0 + yp)) < 1e-15 and delta < 0    # pulled towards bin 7
    P[:] = 1.0
    assert ana.pulse_peak(P)[0] == 0 and ana.pulse_peak(P)[1] == 0.0


@pytest.mark.parametrize("N,m", [(32, 7), (50, 49), (1024, 513)])
def test_bandpass_correction_flattens_an_impulse(N, m):
    """P = delta[b - m]  =>  T[i] = exp(-j 2 pi i m/N); corrected by (m, 0) every B[i] is exactly 1."""
    T = np.array([cmath.exp(-2j * math.pi * ((i * m) % N) / N) for i in range(N)])
    B = ana.bandpass_corrected(T, m, 0.0)
    assert np.abs(B - 1.0).max() < 1e-14
    # a fractional position: half a bin more removes exp(-j pi i / N) as well
    T2 = T * np.array([cmath.exp(-1j * math.pi * i / N) for i in range(N)])
    assert np.abs(ana.bandpass_corrected(T2, m, 0.5) - 1.0).max() < 1e-12


def closed_form_tones(N, n_samples, f_s, f_comb, f_off, t_d, amp):
    """T[i] = (A n_samples / 2) e^{j(phi_i - pi/2)}, phi_i = 2 pi (i f_comb + f_off) t_d, in-band i."""
    T = np.zeros(N, np.complex128)
    first = 0 if f_off else 1
    for i in range(first, N // 2):
        phi = 2 * math.pi * (i * f_comb + f_off) * t_d
        T[i] = 0.5 * amp * n_samples * cmath.exp(1j * (phi - 0.5 * math.pi))
    return T


@pytest.mark.parametrize("f_off,t_d", [(10e3, 5e-9), (10e3, 312.5e-9), (0.0, 12.5e-9), (640e3, 777e-9)])
def test_phase_slope_recovers_the_cable_delay_of_eq21(f_off, t_d):
    f_s, f_comb, N = 32e6, 1e6, 32
    T = closed_form_tones(N, 12800, f_s, f_comb, f_off, t_d, 0.05)
    s, a, rms = ana.phase_slope(T, 0 if f_off else 1, N // 2)
    # slope = 2 pi f_comb t_d; a comb only fixes the delay modulo 1/f_comb, the unwrapped slope picks |t| < 1/(2 f_comb)
    want = ((t_d * f_comb + 0.5) % 1.0 - 0.5) / f_comb
    assert abs(s / (2 * math.pi * f_comb) - want) <= 1e-9 * abs(want)
    want_a = 2 * math.pi * f_off * t_d          # the intercept keeps the true t_d: theta_0 = 2 pi f_off t_d
    assert abs((a - want_a + math.pi) % (2 * math.pi) - math.pi) < 1e-9   # intercept = 2 pi f_off t_d (mod 2 pi)
    assert rms < 1e-9


def test_analyze_on_the_closed_form_pulse_of_eq21():
    """Rotated, folded eq. 2.1 (s = 0): P[b] = (A M / 2j) e^{j w_off D} sum_i e^{j i w_comb (b + D)},
    D = t_d f_s, M = n_samples / N: a Dirichlet kernel whose power peaks at b = -D (mod N)."""
    f_s, f_comb, f_off, N, amp, n_samples = 32e6, 1e6, 10e3, 32, 0.05, 12800
    for t_d in (5e-9, 100e-9, 0.99e-6):
        D = t_d * f_s
        K = N // 2
        P = np.zeros(N, np.complex128)
        for b in range(N):
            acc = 0j
            for i in range(K):
                acc += cmath.exp(2j * math.pi * i * (b + D) / N)
            P[b] = amp * (n_samples / N) / 2j * cmath.exp(2j * math.pi * f_off / f_s * D) * acc
        T = closed_form_tones(N, n_samples, f_s, f_comb, f_off, t_d, amp)
        # the closed-form T is the DFT of the closed-form P (ties the two halves of the pin together)
        Tdft = np.array([sum(P[b] * cmath.exp(-2j * math.pi * ((i * b) % N) / N) for b in range(N)) for i in range(N)])
        assert np.abs(Tdft - T).max() < 1e-9 * np.abs(T).max()
        summary, B = ana.analyze(P, T, f_s, f_comb, f_off)
        true_pos = (-D) % N
        est_pos = (summary[0] + summary[1]) % N
        err = (est_pos - true_pos + N / 2) % N - N / 2
        assert abs(err) < 0.08                     # three-point vertex on a Dirichlet power peak (K = N/2): bias < 0.08 bin
        assert abs(summary[2] - (summary[0] + summary[1]) / f_s) < 1e-18
        assert abs(summary[5] - ((t_d * f_comb + 0.5) % 1.0 - 0.5) / f_comb) <= 1e-9 * t_d
        # corrected by the true position the band-pass phase is flat: arg B[i] = w_off D - pi/2 for every tone
        Bt = ana.bandpass_corrected(T, int(round(true_pos)) % N, true_pos - round(true_pos))
        ph = np.angle(Bt[:K] * cmath.exp(-1j * (2 * math.pi * f_off * t_d - 0.5 * math.pi)))
        assert np.abs(ph).max() < 1e-9
        assert np.allclose(np.abs(B[:K]), 0.5 * amp * n_samples, rtol=1e-12)
