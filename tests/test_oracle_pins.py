"""Pins for the CPU oracle (oracle/pcal_oracle.c) against what the paper and the mathematics fix.

None of these re-type the oracle's formula with the same library call: expected values come from
closed forms derived from eq. 2.1, from exact rational phase arithmetic done with
Python integers, from special cases with textbook answers, or from values the paper prints
(tests/golden/eq2_4_instances.txt).  A dropped term, wrong sign, wrong index or transposed
operand in the oracle fails at least one of them.
"""
import cmath
import math
import os
from fractions import Fraction

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def comb_eq21(n_samples, f_s, f_comb, f_off, t_d, tones, amp=1.0):
    """eq. 2.1 with s[n] = 0, written as the plain sum of sines (fp64)."""
    n = np.arange(n_samples, dtype=np.float64)
    x = np.zeros(n_samples)
    phis = []
    for i in tones:
        w = 2 * math.pi * (i * f_comb + f_off) / f_s
        phi = w * t_d * f_s
        phis.append(phi)
        x += amp * np.sin(w * n + phi)
    return x, np.array(phis)


@pytest.mark.parametrize("f_off,first_tone", [(10e3, 0), (0.0, 1)])
def test_closed_form_eq21(oracle, f_off, first_tone):
    """T[i] = (A N / 2) e^{j(phi_i - pi/2)} for in-band tones, N a multiple of L."""
    f_s, f_comb, t_d = 32e6, 1e6, 5e-9
    nb = 32
    tones = list(range(first_tone, nb // 2))
    N = 12800  # 4 * L, L = 3200
    x, phis = comb_eq21(N, f_s, f_comb, f_off, t_d, tones)
    T = oracle.extract(x, oracle.F64, 1, 0, N, 0, f_s, f_comb, f_off)
    for i, phi in zip(tones, phis):
        amp = 2 * abs(T[i]) / N
        ph = cmath.phase(T[i]) + math.pi / 2
        dphi = (ph - phi + math.pi) % (2 * math.pi) - math.pi
        assert abs(dphi) < 1e-9, (i, dphi)
        assert abs(amp - 1.0) < 1e-9, (i, amp)
    if f_off == 0.0:
        # P real -> T Hermitian; bins 0 and N/2 carry no comb power (sin(0) tone, R5)
        assert abs(T[0]) < 1e-6 and abs(T[nb // 2]) < 1e-6
        for i in tones:
            assert abs(T[nb - i] - T[i].conjugate()) < 1e-6
    else:
        # 2 f_off not a multiple of f_comb -> upper bins empty
        for i in range(nb // 2, nb):
            assert abs(T[i]) < 1e-6, (i, T[i])


def test_closed_form_missing_tone_and_amplitude(oracle):
    f_s, f_comb, f_off, t_d = 16e6, 1e6, 10e3, 12.5e-9
    tones = [1, 2, 5]
    N = 1600 * 3
    x, phis = comb_eq21(N, f_s, f_comb, f_off, t_d, tones, amp=0.25)
    T = oracle.extract(x, oracle.F64, 1, 0, N, 0, f_s, f_comb, f_off)
    for i in range(8):
        if i in tones:
            assert abs(2 * abs(T[i]) / N - 0.25) < 1e-9
        else:
            assert abs(T[i]) < 1e-6


def exact_phasor(n, F, Fs):
    """exp(-j 2 pi (n F mod Fs)/Fs) with the reduction done in Python integers / Fractions."""
    frac = Fraction((n * F) % Fs, Fs)
    return cmath.exp(-2j * math.pi * float(frac))


@pytest.mark.parametrize("n1", [0, 1, 37, 3199, 3200, 123457])
def test_impulse_pins_phase_origin_and_bin_index(oracle, n1):
    """x = delta[n - n1]  =>  T[i] = e^{-j (i w_comb + w_off) n1} exactly (R8)."""
    f_s, f_comb, f_off = 32e6, 1e6, 10e3
    Fs, Fc, Fo = 32_000_000_000_000, 1_000_000_000_000, 10_000_000_000
    N = n1 + 5
    x = np.zeros(N)
    x[n1] = 1.0
    T = oracle.extract(x, oracle.F64, 1, 0, N, 0, f_s, f_comb, f_off)
    for i in range(32):
        want = exact_phasor(n1, i * Fc + Fo, Fs)
        assert abs(T[i] - want) < 1e-12, (i, T[i], want)
    # same impulse delivered as a later segment: absolute index = n_abs0 + m
    y = np.zeros(5)
    y[2] = 1.0
    T2 = oracle.extract(y, oracle.F64, 1, 0, 5, n1 - 2 if n1 >= 2 else 0, f_s, f_comb, f_off)
    if n1 >= 2:
        assert np.max(np.abs(T2 - T)) < 1e-12


@pytest.mark.parametrize("N", [4096, 4109])
def test_fold_dft_equals_bruteforce_per_tone_correlation(oracle, N):
    """fold + DFT == per-tone correlation, any length."""
    rng = np.random.RandomState(7)
    x = rng.standard_normal(N)
    f_s, f_comb, f_off = 32e6, 1e6, 10e3
    Fs, Fc, Fo = 32_000_000_000_000, 1_000_000_000_000, 10_000_000_000
    T_fold = oracle.extract(x, oracle.F64, 1, 0, N, 0, f_s, f_comb, f_off)
    T_dir = oracle.direct(x, oracle.F64, 1, 0, 0, N, 0, f_s, f_comb, f_off)
    # independent brute force: exact integer phase in Python, numpy only for the final dot
    for i in [0, 1, 7, 16, 31]:
        F = i * Fc + Fo
        ph = np.array([((n * F) % Fs) / Fs for n in range(N)], dtype=np.float64)
        want = np.dot(x, np.cos(2 * math.pi * ph)) - 1j * np.dot(x, np.sin(2 * math.pi * ph))
        assert abs(T_dir[i] - want) < 1e-9
        assert abs(T_fold[i] - want) < 1e-9
    assert np.max(np.abs(T_fold - T_dir)) < 1e-9


def test_split_point_invariance(oracle):
    rng = np.random.RandomState(11)
    N = 10007
    x = rng.standard_normal(N)
    f = (32e6, 1e6, 10e3)
    pr, pi = oracle.fold_ld(x, oracle.F64, 1, 0, 0, 1, N, 0, *f)
    for cuts in ([1], [4096], [17, 3200, 9999]):
        qr = np.zeros(32, np.longdouble)
        qi = np.zeros(32, np.longdouble)
        edges = [0] + cuts + [N]
        for a, b in zip(edges[:-1], edges[1:]):
            seg = np.ascontiguousarray(x[a:b])
            r, i = oracle.fold_ld(seg, oracle.F64, 1, 0, 0, 1, b - a, a, *f)
            qr += r
            qi += i
        assert float(np.max(np.abs(qr - pr))) < 1e-11 and float(np.max(np.abs(qi - pi))) < 1e-11
    # integer path: bit-identical
    xi = rng.randint(-127, 128, size=N).astype(np.int8)
    whole = oracle.fold_i64(xi, oracle.I8, 1, 0, 0, 1, N, 5, 32)
    a = oracle.fold_i64(np.ascontiguousarray(xi[:4001]), oracle.I8, 1, 0, 0, 1, 4001, 5, 32)
    b = oracle.fold_i64(np.ascontiguousarray(xi[4001:]), oracle.I8, 1, 0, 0, 1, N - 4001, 5 + 4001, 32)
    assert np.array_equal(whole, a + b)
    # brute force of the integer fold
    want = np.zeros(32, np.int64)
    for m in range(N):
        want[(5 + m) % 32] += int(xi[m])
    assert np.array_equal(whole, want)


def test_constant_input_and_hermitian(oracle):
    N = 32 * 50
    x = np.ones(N)
    T = oracle.extract(x, oracle.F64, 1, 0, N, 0, 32e6, 1e6, 0.0)
    assert abs(T[0] - N) < 1e-9
    assert np.max(np.abs(T[1:])) < 1e-9
    rng = np.random.RandomState(3)
    y = rng.standard_normal(1000)
    pr, pi = oracle.fold_ld(y, oracle.F64, 1, 0, 0, 1, 1000, 0, 32e6, 1e6, 0.0)
    assert float(np.max(np.abs(pi))) == 0.0  # P purely real without rotation
    T = oracle.dft(pr, pi)
    for i in range(1, 32):
        assert abs(T[32 - i] - T[i].conjugate()) < 1e-10


def test_dft_against_textbook_cases(oracle):
    """DFT(delta[b-b0]) = e^{-j 2 pi i b0/N}; DFT(e^{+j 2 pi k b/N}) = N delta[i-k]; numpy fft."""
    N = 64
    p = np.zeros(N)
    p[5] = 1.0
    T = oracle.dft(p, np.zeros(N))
    for i in range(N):
        assert abs(T[i] - cmath.exp(-2j * math.pi * i * 5 / N)) < 1e-14
    b = np.arange(N)
    z = np.exp(2j * math.pi * 3 * b / N)
    T = oracle.dft(z.real, z.imag)
    want = np.zeros(N, complex)
    want[3] = N
    assert np.max(np.abs(T - want)) < 1e-12
    rng = np.random.RandomState(5)
    for n in (12, 100, 512):  # non-power-of-two too
        z = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        assert np.max(np.abs(oracle.dft(z.real, z.imag) - np.fft.fft(z))) < 1e-11 * n


def test_rotator_length_paper_instances(oracle):
    for line in open(os.path.join(GOLD, "eq2_4_instances.txt")):
        if line.startswith("#") or not line.strip():
            continue
        f_s, f_comb, f_off, nb, nrot = [int(t) for t in line.split()[:5]]
        assert oracle.rotator_len(f_s, f_off) == nrot
        assert oracle.to_uhz(f_s) // oracle.to_uhz(f_comb) == nb
    # R6: N_rotator need not be a multiple of N_bins (32 MHz / 640 kHz -> 50)
    assert oracle.rotator_len(32e6, 640e3) == 50
    assert oracle.rotator_len(32e6, 0.0) == 1
    # R16: 1234.567 Hz at 1024 MHz is co-prime on the micro-hertz grid up to a small factor
    assert oracle.rotator_len(1024e6, 1234.567) == 1_024_000_000_000_000 // math.gcd(1_024_000_000_000_000, 1_234_567_000)


def test_phase_reduction_is_exact_for_huge_indices(oracle):
    L = oracle.lib()
    Fs, F = 1_024_000_000_000_000, 1_234_567_000
    for n in (0, 1, 2**16, 4_000_000_000 - 1, 2**63 + 12345):
        assert L.orc_phase_num(n, F, Fs) == (n * F) % Fs


def test_decode_tables_and_packing(oracle):
    """DESIGN.md R15: hand-built words; the table look-up is the whole definition."""
    byte = np.array([0b11100100, 0b00011011], dtype=np.uint8)  # codes 0,1,2,3 then 3,2,1,0 (LSB first)
    ob = [oracle.decode(byte, oracle.TWO_BIT_OFFSET_BINARY, 1, 0, m) for m in range(8)]
    sm = [oracle.decode(byte, oracle.TWO_BIT_SIGN_MAG, 1, 0, m) for m in range(8)]
    assert ob == [-3, -1, 1, 3, 3, 1, -1, -3]
    assert sm == [1, 3, -1, -3, -3, -1, 3, 1]
    # 16 channels per little-endian uint32, channel c in bits 2c..2c+1
    words = np.array([3 << 10, (1 << 30) | 2], dtype=np.uint32)
    for c in range(16):
        v0 = oracle.decode(words, oracle.TWO_BIT_OFFSET_BINARY, 16, c, 0)
        assert v0 == (3 if c == 5 else -3)
    assert oracle.decode(words, oracle.TWO_BIT_SIGN_MAG, 16, 15, 1) == 3   # code 1 -> +3
    assert oracle.decode(words, oracle.TWO_BIT_SIGN_MAG, 16, 0, 1) == -1   # code 2 -> -1
    assert oracle.decode(words, oracle.TWO_BIT_SIGN_MAG, 16, 7, 1) == 1    # code 0 -> +1
    i8 = np.array([-128, -1, 0, 127], dtype=np.int8)
    assert [oracle.decode(i8, oracle.I8, 1, 0, m) for m in range(4)] == [-128, -1, 0, 127]
    f32 = np.array([1.5, -2.25], dtype=np.float32)
    assert [oracle.decode(f32, oracle.F32, 1, 0, m) for m in range(2)] == [1.5, -2.25]


def test_k_shift_is_a_bin_rotation(oracle):
    """rotating by w_off + k w_comb circularly shifts the DFT bins by k."""
    rng = np.random.RandomState(9)
    N = 3203
    x = rng.standard_normal(N)
    T = oracle.extract(x, oracle.F64, 1, 0, N, 0, 32e6, 1e6, 10e3)
    k = 8
    Tk = oracle.extract(x, oracle.F64, 1, 0, N, 0, 32e6, 1e6, 10e3 + k * 1e6)
    for i in range(32):
        assert abs(Tk[(i - k) % 32] - T[i]) < 1e-10


def test_linearity_and_tabulated_variant(oracle):
    rng = np.random.RandomState(13)
    N = 7000
    x = rng.standard_normal(N)
    y = rng.standard_normal(N)
    f = (16e6, 1e6, 10e3)
    Tx = oracle.extract(x, oracle.F64, 1, 0, N, 3, *f)
    Ty = oracle.extract(y, oracle.F64, 1, 0, N, 3, *f)
    Tz = oracle.extract(2.0 * x - 0.5 * y, oracle.F64, 1, 0, N, 3, *f)
    assert np.max(np.abs(Tz - (2.0 * Tx - 0.5 * Ty))) < 1e-10
    Tt = oracle.extract(x, oracle.F64, 1, 0, N, 3, *f, tabulated=True)
    assert np.max(np.abs(Tt - Tx)) < 1e-11
    Tp = oracle.extract(x, oracle.F64, 1, 0, N, 3, *f, threads=3)
    assert np.max(np.abs(Tp - Tx)) < 1e-11
    # strided visit (one bin only) equals that bin of the full fold
    pr, pi = oracle.fold_ld(x, oracle.F64, 1, 0, 0, 1, N, 3, *f)
    b = 5
    m_first = (b - 3) % 16
    qr, qi = oracle.fold_ld(x, oracle.F64, 1, 0, m_first, 16, N, 3, *f)
    assert abs(float(qr[b] - pr[b])) < 1e-12 and abs(float(qi[b] - pi[b])) < 1e-12
    assert float(np.sum(np.abs(qr))) == abs(float(qr[b]))
