// pcal_genstudy.cuh -- accuracy of the paper's sinewave generators over many cycles.
//
// PAPER.md:74-101 (eq. 2.6: Coupled Form, Magic Circle, Direct Form 2nd Order Resonator; eq. 2.7:
// the DFR as one fused multiply-add), PAPER.md:142-153 (direct method: trig of a running float32
// phase), PAPER.md:97 (k-shift: rotate at w_offset + k w_comb), PAPER.md:505 (the accuracy
// comparison whose figure is missing from the text).  One thread runs one (form, precision,
// frequency) case for n_steps samples and records, per checkpoint interval, the largest distance
// between the generated phasor and exp(-j n dphi) evaluated from the exactly reduced integer phase.
// Every operation of a recursion is a single correctly rounded fp32 / fp64 instruction
// (__fmul_rn ... : no contraction), in the order the equations are written.  Readings: DESIGN.md R26.
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include "pcal_common.cuh"

namespace pcal {

enum GenForm : int { GEN_CFO = 0, GEN_MCO = 1, GEN_DFR = 2, GEN_DFR_FMA = 3, GEN_DIRECT = 4 };

struct GenStudyCase {
    int32_t form, precision;      // GenForm; 32 or 64
    uint64_t Fs, F;               // micro-hertz: sample rate, rotator frequency
    double cn, sn, eps, two_c;    // cos(dphi), sin(dphi), 2 sin(dphi/2), 2 cos(dphi)   (fp64, host libm)
    double s_half;                // sin(dphi/2): Magic Circle start value
    float dphi32;                 // float32(dphi): the direct method's phase increment
};

template <typename T> struct Rn;
template <> struct Rn<float> {
    static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
    static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
    static __device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
    static __device__ __forceinline__ float fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
};
template <> struct Rn<double> {
    static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
    static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
    static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
    static __device__ __forceinline__ double fma(double a, double b, double c) { return __fma_rn(a, b, c); }
};

template <typename T>
__device__ void gen_study_run(const GenStudyCase& C, uint64_t n_steps, uint32_t n_chk, double* err) {
    using R = Rn<T>;
    const T cn = (T)C.cn, sn = (T)C.sn, eps = (T)C.eps, two_c = (T)C.two_c;
    T y1 = (T)1.0, y2 = C.form == GEN_MCO ? (T)(-C.s_half) : (T)0.0;       // CFO / MCO state
    T c_prev = (T)1.0, c_cur = cn, s_prev = (T)0.0, s_cur = (T)(-C.sn);     // DFR: cos and -sin sequences
    uint64_t k = 0, k2 = C.F % (2 * C.Fs);          // (n F) mod Fs ; ((2n+1) F) mod 2Fs
    const uint64_t two_F = (2 * C.F) % (2 * C.Fs);
    for (uint64_t n = 1; n <= n_steps; ++n) {
        T o1, o2;
        if (C.form == GEN_CFO) {
            const T n1 = R::add(R::mul(cn, y1), R::mul(sn, y2));
            const T n2 = R::add(R::mul(-sn, y1), R::mul(cn, y2));
            y1 = n1; y2 = n2; o1 = y1; o2 = y2;
        } else if (C.form == GEN_MCO) {
            y1 = R::add(y1, R::mul(eps, y2));
            y2 = R::add(R::mul(-eps, y1), y2);       // the updated y1 (R26)
            o1 = y1; o2 = y2;
        } else if (C.form == GEN_DFR || C.form == GEN_DFR_FMA) {
            if (n >= 2) {
                T nc, ns;
                if (C.form == GEN_DFR) { nc = R::sub(R::mul(two_c, c_cur), c_prev); ns = R::sub(R::mul(two_c, s_cur), s_prev); }
                else { nc = R::fma(two_c, c_cur, -c_prev); ns = R::fma(two_c, s_cur, -s_prev); }
                c_prev = c_cur; c_cur = nc; s_prev = s_cur; s_cur = ns;
            }
            o1 = c_cur; o2 = s_cur;
        } else {                                       // direct method, listing K1, sign of eq. 2.3
            const float ph = __fmul_rn((float)n, C.dphi32);
            o1 = (T)cosf(ph); o2 = (T)(-sinf(ph));
        }
        k += C.F; if (k >= C.Fs) k -= C.Fs;
        k2 += two_F; if (k2 >= 2 * C.Fs) k2 -= 2 * C.Fs;
        double es, ec;
        sincospi(2.0 * ((double)k / (double)C.Fs), &es, &ec);
        double ei = -es;
        if (C.form == GEN_MCO) ei = -sinpi((double)k2 / (double)C.Fs);      // -sin((n + 1/2) dphi)
        const double d = hypot((double)o1 - ec, (double)o2 - ei);
        uint64_t j = (n - 1) * n_chk / n_steps;
        if (j >= n_chk) j = n_chk - 1;
        if (d > err[j]) err[j] = d;
    }
}

__global__ void gen_study_kernel(const GenStudyCase* cases, uint32_t n_cases, uint64_t n_steps, uint32_t n_chk, double* err) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_cases) return;
    double* e = err + (size_t)t * n_chk;
    for (uint32_t j = 0; j < n_chk; ++j) e[j] = 0.0;
    const GenStudyCase C = cases[t];
    if (C.precision == 32) gen_study_run<float>(C, n_steps, n_chk, e);
    else gen_study_run<double>(C, n_steps, n_chk, e);
}

}  // namespace pcal
