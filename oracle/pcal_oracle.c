/*
 * pcal_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the multi-tone phase-calibration (PCal)
 * extraction hot path of Wagner & Pogrebenko, "Fast Multi-tone Phase Calibration Signal
 * Extraction" (/root/reference/PAPER.md, cited below as PAPER.md:<line>).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call into this file.  It shares no code, header, table or constant with the CUDA path under
 * paper_2501_05993_b200/csrc/ and neither includes the other.
 *
 * What it computes; every function states the passage it follows:
 *   orc_decode      sample decode table (2-bit / int8 / float32)        PAPER.md:31 + DESIGN.md R15
 *   orc_phase_num   (n*F) mod F_s in exact integers                      eq. 2.3/2.5
 *   orc_direct      T[i] = sum_n v[n] exp(-j(i w_comb + w_off) n)        eq. 2.1-2.3
 *   orc_fold        P[b] = sum_{n = b mod N_bins} v[n] exp(-j w_off n)   eq. 2.3 then 2.2
 *   orc_fold_i64    P[b] exact int64 when w_off = 0 and integer samples  eq. 2.2
 *   orc_dft         T[i] = sum_b P[b] exp(-j 2 pi i b / N_bins)          "DFT(P)"
 *   orc_rotator_len N_rotator = f_s / gcd(f_s, f_offset)                 eq. 2.4
 *
 * Arithmetic: sample index times frequency is formed in unsigned __int128 and reduced modulo
 * F_s BEFORE any conversion to floating point (this removes the accuracy decline with n that
 * PAPER.md:142 warns about); phasors from glibc sincos() on the reduced phase (fp64, < 1 ulp);
 * all sums are carried in x87 long double (64-bit mantissa).  No blocking, no fusion, no
 * reordering: one loop over the samples in index order.
 *
 * Frequencies are integers on a 1 micro-hertz grid (reading R16).
 * Sign conventions (R1, R3): rotator exp(-j ...) as eq. 2.3 states; forward,
 * unnormalised DFT.
 *
 * Pins (tests/test_oracle_pins.py): closed form of eq. 2.1 with s[n]=0, impulse response,
 * brute force in exact rational phase arithmetic (Python ints + mpmath-free Fraction reduction),
 * split-point invariance, constant input, Hermitian symmetry, eq. 2.4's printed instance
 * (16 MHz / 10 kHz -> 1600), hand-built packed words.
 * Unpinned by the paper (defined in DESIGN.md R15-R17): the 2-bit code->level tables, the
 * micro-hertz snapping and the tolerance denominator -- "parity unpinned" for those three
 * definitions only; the tables are still pinned to DESIGN.md's statement by hand-built words.
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stddef.h>

typedef unsigned __int128 u128;

/* sample formats (oracle-private numbering) */
enum { ORC_F32 = 0, ORC_I8 = 1, ORC_2BIT_OFFSET_BINARY = 2, ORC_2BIT_SIGN_MAG = 3,
       ORC_F64 = 4 /* oracle-only: fp64 samples, so the closed-form pin is not limited by a float32 cast */ };

/* DESIGN.md R15: OFFSET_BINARY code c -> 2c-3 ; SIGN_MAG code=(s<<1)|m, s=1 negative, m=1 -> |3| */
static const double LEVEL_OB[4] = { -3.0, -1.0, +1.0, +3.0 };
static const double LEVEL_SM[4] = { +1.0, +3.0, -1.0, -3.0 };

/*
 * Value of sample m (0-based within buf) of channel c.
 *  - float32: buf is float[ ], single channel.
 *  - int8: buf is int8_t[ ], single channel, two's complement.
 *  - 2-bit, n_channels == 1: 4 samples per byte, sample m in bits 2(m&3)..2(m&3)+1 of byte m>>2
 *    (LSB first, BASELINE.json config 2).
 *  - 2-bit, n_channels == C > 1 (C*2 <= 32): one little-endian word of C*2 bits per time sample,
 *    channel c in bits 2c..2c+1 (BASELINE.json config 4); words are packed back to back.
 */
double orc_decode(const void *buf, int fmt, int n_channels, int c, uint64_t m)
{
    if (fmt == ORC_F32) return (double)((const float *)buf)[m];
    if (fmt == ORC_F64) return ((const double *)buf)[m];
    if (fmt == ORC_I8) return (double)((const int8_t *)buf)[m];
    const uint8_t *b = (const uint8_t *)buf;
    uint64_t bitpos = (n_channels == 1) ? 2 * m : (m * (uint64_t)n_channels + (uint64_t)c) * 2;
    unsigned code = (b[bitpos >> 3] >> (bitpos & 7)) & 3u;
    return (fmt == ORC_2BIT_OFFSET_BINARY) ? LEVEL_OB[code] : LEVEL_SM[code];
}

/* (n * F) mod Fs, exact.  n < 2^64, F < 2^64 -> product < 2^128. */
uint64_t orc_phase_num(uint64_t n, uint64_t F, uint64_t Fs)
{
    return (uint64_t)(((u128)n * (u128)F) % (u128)Fs);
}

static uint64_t gcd_u64(uint64_t a, uint64_t b)
{
    while (b) { uint64_t t = a % b; a = b; b = t; }
    return a;
}

/* eq. 2.4: N_rotator = f_s / gcd(f_s, f_offset); f_offset = 0 -> 1 */
uint64_t orc_rotator_len(uint64_t Fs, uint64_t Foff)
{
    return Fs / gcd_u64(Fs, Foff);
}

/* exp(-j 2 pi k / Fs) for an exactly reduced numerator k in [0, Fs) */
static void phasor_neg(uint64_t k, uint64_t Fs, double *c, double *s)
{
    double ang = (double)(2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)Fs);
    double sn, cs;
    sincos(ang, &sn, &cs);
    *c = cs;
    *s = -sn;
}

/*
 * O-direct (north_star; eq. 2.1-2.3 combined):
 *   T[i] += sum_{m=m0}^{m0+count-1} v[m] * exp(-j 2 pi ((n (i Fcomb + Foff)) mod Fs) / Fs),
 *   n = n_abs0 + m   (absolute sample index since the last reset, R8),
 *   i = 0..N_bins-1, N_bins = Fs / Fcomb.
 * T_re/T_im are long double[N_bins], accumulated into (caller zeroes them).  O(count * N_bins).
 */
void orc_direct(const void *buf, int fmt, int n_channels, int c,
                uint64_t m0, uint64_t count, uint64_t n_abs0,
                uint64_t Fs, uint64_t Fcomb, uint64_t Foff,
                long double *T_re, long double *T_im)
{
    uint64_t n_bins = Fs / Fcomb;
    for (uint64_t m = m0; m < m0 + count; m++) {
        double v = orc_decode(buf, fmt, n_channels, c, m);
        uint64_t n = n_abs0 + m;
        for (uint64_t i = 0; i < n_bins; i++) {
            /* tone frequency i*Fcomb + Foff, reduced mod Fs first (exp is Fs-periodic in it) */
            uint64_t Ftone = (uint64_t)(((u128)i * Fcomb + Foff) % Fs);
            double cs, sn;
            phasor_neg(orc_phase_num(n, Ftone, Fs), Fs, &cs, &sn);
            T_re[i] += (long double)v * (long double)cs;
            T_im[i] += (long double)v * (long double)sn;
        }
    }
}

/*
 * O-fold, first half (eq. 2.3 then eq. 2.2):
 *   P[b] += sum over m = m_first, m_first+m_step, ... < m_end of
 *           v[m] * exp(-j 2 pi ((n Foff) mod Fs) / Fs),  n = n_abs0 + m,  b = n mod N_bins.
 * m_step = 1 is the whole stream; m_step = N_bins visits the samples of one bin only (used to
 * check sampled bins of a multi-gigasample run).  P_re/P_im are long double[N_bins].
 */
void orc_fold(const void *buf, int fmt, int n_channels, int c,
              uint64_t m_first, uint64_t m_step, uint64_t m_end, uint64_t n_abs0,
              uint64_t Fs, uint64_t Fcomb, uint64_t Foff,
              long double *P_re, long double *P_im)
{
    uint64_t n_bins = Fs / Fcomb;
    for (uint64_t m = m_first; m < m_end; m += m_step) {
        double v = orc_decode(buf, fmt, n_channels, c, m);
        uint64_t n = n_abs0 + m;
        double cs = 1.0, sn = 0.0;
        if (Foff != 0) phasor_neg(orc_phase_num(n, Foff, Fs), Fs, &cs, &sn);
        uint64_t b = n % n_bins;
        P_re[b] += (long double)v * (long double)cs;
        P_im[b] += (long double)v * (long double)sn;
    }
}

/*
 * O-fold with the rotator tabulated (eq. 2.4): for a rational offset the phasor
 * takes only N_rotator distinct values, phasor[n mod N_rotator]; this variant looks them up in a
 * table built with the very same phasor_neg() -- identical values, not an approximation
 * (SURVEY.md section 8(c)).  table_c/table_s are caller-provided scratch of N_rotator doubles.
 */
void orc_fold_tabulated(const void *buf, int fmt, int n_channels, int c,
                        uint64_t m_first, uint64_t m_step, uint64_t m_end, uint64_t n_abs0,
                        uint64_t Fs, uint64_t Fcomb, uint64_t Foff,
                        double *table_c, double *table_s,
                        long double *P_re, long double *P_im)
{
    uint64_t n_bins = Fs / Fcomb;
    uint64_t n_rot = orc_rotator_len(Fs, Foff);
    for (uint64_t r = 0; r < n_rot; r++)
        phasor_neg(orc_phase_num(r, Foff, Fs), Fs, &table_c[r], &table_s[r]);
    for (uint64_t m = m_first; m < m_end; m += m_step) {
        double v = orc_decode(buf, fmt, n_channels, c, m);
        uint64_t n = n_abs0 + m;
        uint64_t r = n % n_rot;
        uint64_t b = n % n_bins;
        P_re[b] += (long double)v * (long double)table_c[r];
        P_im[b] += (long double)v * (long double)table_s[r];
    }
}

/*
 * O-int (eq. 2.2 with Foff = 0 on integer samples): exact int64 bins.
 * Returns -1 if fmt is float32 (not an integer input), else 0.
 */
int orc_fold_i64(const void *buf, int fmt, int n_channels, int c,
                 uint64_t m_first, uint64_t m_step, uint64_t m_end, uint64_t n_abs0,
                 uint64_t n_bins, int64_t *P)
{
    if (fmt == ORC_F32 || fmt == ORC_F64) return -1;
    for (uint64_t m = m_first; m < m_end; m += m_step) {
        int64_t v = (int64_t)orc_decode(buf, fmt, n_channels, c, m);
        P[(n_abs0 + m) % n_bins] += v;
    }
    return 0;
}

/*
 * O-fold, second half ("DFT(P)"; forward, unnormalised, R3):
 *   T[i] = sum_{b=0}^{N-1} P[b] * exp(-j 2 pi ((i b) mod N) / N).
 * Twiddle index reduced in integers; trigonometry and sums in long double.
 * T is double[2*N] (re, im interleaved).
 */
void orc_dft(const long double *P_re, const long double *P_im, uint64_t N, double *T)
{
    for (uint64_t i = 0; i < N; i++) {
        long double ar = 0.0L, ai = 0.0L;
        for (uint64_t b = 0; b < N; b++) {
            uint64_t k = (uint64_t)(((u128)i * b) % N);
            long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)N;
            long double cs = cosl(ang), sn = -sinl(ang);
            ar += P_re[b] * cs - P_im[b] * sn;
            ai += P_re[b] * sn + P_im[b] * cs;
        }
        T[2 * i] = (double)ar;
        T[2 * i + 1] = (double)ai;
    }
}
