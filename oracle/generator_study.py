"""TEST INFRASTRUCTURE, NOT THE PRODUCT -- step-by-step emulation of the paper's sinewave generators.

SURVEY.md section 8(f)2 / PAPER.md:74-101, 142, 505: the accuracy of the recursive oscillators
(eq. 2.6: Coupled Form, Magic Circle, Direct Form 2nd Order Resonator; eq. 2.7: the DFR as one
fused multiply-add) and of the direct method (listing K1: trig of a running fp32
phase) over many cycles, against the exact phasor exp(-j n dphi) whose phase (n F_offset) mod F_s
is reduced in Python integers.  Every arithmetic operation is rounded once to the stated precision
(numpy float32 / Python float), in the order the equations are written; the fused multiply-add is
rounded exactly from rationals.  Pure-Python loops: small n only.

Readings (R26): the rotation is exp(-j n dphi) (R1), so the sine outputs start at
-sin(dphi); the Magic Circle's second line uses the UPDATED y1[n] (as printed, with y1[n-1] twice,
the recursion spirals outwards and could not be "numerically ideal"); started from
(1, -sin(dphi/2)) -- the paper gives no initial values -- its outputs are cos(n dphi) and
-sin((n + 1/2) dphi), the half-step offset inherent in that form.
Shares no code with paper_2501_05993_b200/.  Pins: tests/test_generator_study_pins.py.
"""
from __future__ import annotations

import math
from fractions import Fraction

import numpy as np

CFO, MCO, DFR, DFR_FMA, DIRECT = 0, 1, 2, 3, 4


def _round_to(x: Fraction, bits: int) -> float:
    """Nearest value with a `bits`-bit significand, ties to even (no subnormals/overflow needed here)."""
    if x == 0:
        return 0.0
    sign = -1 if x < 0 else 1
    a = -x if x < 0 else x
    e = a.numerator.bit_length() - a.denominator.bit_length()
    if Fraction(2) ** e > a:
        e -= 1                                   # 2^e <= a < 2^(e+1)
    q = a / Fraction(2) ** (e - (bits - 1))      # in [2^(bits-1), 2^bits)
    m = q.numerator // q.denominator
    rem = q - m
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (m & 1)):
        m += 1
    return sign * float(Fraction(m) * Fraction(2) ** (e - (bits - 1)))


class _Arith:
    """mul / add / sub / fma rounded once to float32 (bits=24) or float64 (bits=53)."""

    def __init__(self, precision: int):
        self.bits = 24 if precision == 32 else 53
        self.t = np.float32 if precision == 32 else np.float64

    def c(self, x):
        return self.t(x)

    def mul(self, a, b):
        return self.t(a) * self.t(b)

    def add(self, a, b):
        return self.t(a) + self.t(b)

    def sub(self, a, b):
        return self.t(a) - self.t(b)

    def fma(self, a, b, c):
        return self.t(_round_to(Fraction(float(a)) * Fraction(float(b)) + Fraction(float(c)), self.bits))


def exact_phasor(n: int, F_uhz: int, Fs_uhz: int):
    """exp(-j 2 pi ((n F) mod Fs)/Fs) with the phase reduced in integers."""
    k = (n * F_uhz) % Fs_uhz
    ang = 2.0 * math.pi * (k / Fs_uhz)
    return math.cos(ang), -math.sin(ang)


def run(form: int, precision: int, f_s_hz: float, f_rot_hz: float, n_steps: int, n_chk: int):
    """max_n |y[n] - exact[n]| over each of n_chk equal intervals of n = 1..n_steps (fp64), where
    y = y1 + j y2 of the chosen recursion rotating at f_rot (= f_offset + k f_comb for a k-shift)."""
    Fs, F = int(round(f_s_hz * 1e6)), int(round(f_rot_hz * 1e6))
    dphi = 2.0 * math.pi * F / Fs                      # eq. 2.5 (fp64 constant, then rounded to the precision)
    A = _Arith(precision)
    cn, sn = A.c(math.cos(dphi)), A.c(math.sin(dphi))
    eps = A.c(2.0 * math.sin(0.5 * dphi))
    two_c = A.c(2.0 * math.cos(dphi))
    err = [0.0] * n_chk
    # states
    if form == CFO:
        y1, y2 = A.c(1.0), A.c(0.0)
    elif form == MCO:
        y1, y2 = A.c(1.0), A.c(-math.sin(0.5 * dphi))   # so that y1[n] = cos(n dphi) exactly (R26)
    elif form in (DFR, DFR_FMA):
        c_prev, c_cur = A.c(1.0), cn                   # cos(0), cos(dphi)
        s_prev, s_cur = A.c(0.0), A.c(-math.sin(dphi))  # -sin(0), -sin(dphi)
    dphi32 = np.float32(dphi)
    for n in range(1, n_steps + 1):
        half_step = False
        if form == CFO:
            n1 = A.add(A.mul(cn, y1), A.mul(sn, y2))
            n2 = A.add(A.mul(-sn, y1), A.mul(cn, y2))
            y1, y2 = n1, n2
            o1, o2 = y1, y2
        elif form == MCO:
            y1 = A.add(y1, A.mul(eps, y2))
            y2 = A.add(A.mul(-eps, y1), y2)             # updated y1 (R26)
            o1, o2 = y1, y2
            half_step = True
        elif form in (DFR, DFR_FMA):
            if n >= 2:
                if form == DFR:
                    nc = A.sub(A.mul(two_c, c_cur), c_prev)
                    ns = A.sub(A.mul(two_c, s_cur), s_prev)
                else:
                    nc = A.fma(two_c, c_cur, -c_prev)
                    ns = A.fma(two_c, s_cur, -s_prev)
                c_prev, c_cur, s_prev, s_cur = c_cur, nc, s_cur, ns
            o1, o2 = c_cur, s_cur
        else:                                          # DIRECT, listing K1 with the sign of eq. 2.3
            ph = np.float32(n) * dphi32                 # running phase in float32
            o1, o2 = np.cos(ph, dtype=np.float32), -np.sin(ph, dtype=np.float32)
        er, ei = exact_phasor(n, F, Fs)
        if half_step:                                   # -sin((n + 1/2) dphi): phase (2n+1) F / (2 Fs)
            k2 = ((2 * n + 1) * F) % (2 * Fs)
            ei = -math.sin(2.0 * math.pi * (k2 / (2 * Fs)))
        d = math.hypot(float(o1) - er, float(o2) - ei)
        j = min(n_chk - 1, (n - 1) * n_chk // n_steps)
        if d > err[j]:
            err[j] = d
    return np.array(err)
