// pcal_analysis.cuh -- PCal data analysis on the device.
//
// "Each of the bin i in P[i] ... correspond to a time domain delay t_d(i) = i/f_s.
// The original average delay t_d can be recovered using for example a hyperbolic estimate across
// the neighboring bins around the largest component."  PAPER.md:134-136: group delay "as the
// position of the maximum power", then the "group delay corrected band pass profile".
// PAPER.md:39-42 (eq. 2.1): phi_i = (i w_comb + w_offset) t_d f_s, so the tone phases are linear in
// the tone index with slope 2 pi f_comb t_d.
// Readings (R23-R25): three-point vertex on the power envelope |P|^2 with cyclic
// neighbours; phases unwrapped sequentially (every step wrapped into [-pi, pi)); unweighted least
// squares with a free intercept over the in-band tones.
//
// One CTA per channel.  Decisions that produce integers (the arg-max bin, the 2 pi unwrapping) are
// taken in fp64 with un-contracted multiplies/adds, the same arithmetic an fp64 CPU evaluation
// uses, so they agree with it bit for bit; sums that feed only floating-point outputs use fixed
// trees.  Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include "pcal_common.cuh"

namespace pcal {

constexpr int kAnaThreads = 256;
constexpr int kNSummary = 8;   // == PCAL_N_SUMMARY

struct AnalyzeParams {
    const double2* P;        // [device] folded bins [C][N]
    const double2* T;        // [device] tone spectrum [C][N], natural order
    double* summary;         // [device] [C][kNSummary]
    double2* B;              // [device] [C][N] group-delay corrected band-pass
    double f_s_hz, f_comb_hz;
    uint32_t N;
    uint32_t zero_offset_mask;   // bit c set: channel c has f_offset == 0 (tone 0 is sin(0) = 0)
};

__global__ void __launch_bounds__(kAnaThreads) analyze_kernel(AnalyzeParams A) {
    extern __shared__ double ana_sm[];          // [N] power, then [K] unwrapped phases
    __shared__ double s_val[kAnaThreads];
    __shared__ uint32_t s_idx[kAnaThreads];
    __shared__ double s_sum[kAnaThreads];
    __shared__ double s_pos[2];                 // b*, delta
    const uint32_t c = blockIdx.x, tid = threadIdx.x, N = A.N;
    const double2* P = A.P + (size_t)c * N;
    const double2* T = A.T + (size_t)c * N;

    // ---- power envelope, its maximum (first index on ties) and its sum ----
    double best = -1.0, part = 0.0;
    uint32_t best_i = 0;
    for (uint32_t b = tid; b < N; b += kAnaThreads) {
        const double2 p = P[b];
        const double w = __dadd_rn(__dmul_rn(p.x, p.x), __dmul_rn(p.y, p.y));
        ana_sm[b] = w;
        part += w;
        if (w > best) { best = w; best_i = b; }      // ascending b: keeps the first of equal values
    }
    s_val[tid] = best; s_idx[tid] = best_i; s_sum[tid] = part;
    __syncthreads();
    for (uint32_t s = kAnaThreads / 2; s > 0; s >>= 1) {
        if (tid < s) {
            const double v = s_val[tid + s];
            const uint32_t i = s_idx[tid + s];
            if (v > s_val[tid] || (v == s_val[tid] && i < s_idx[tid])) { s_val[tid] = v; s_idx[tid] = i; }
            s_sum[tid] += s_sum[tid + s];
        }
        __syncthreads();
    }
    if (tid == 0) {
        const uint32_t bs = s_idx[0];
        const double ym = ana_sm[(bs + N - 1) % N], y0 = ana_sm[bs], yp = ana_sm[(bs + 1) % N];
        const double denom = __dadd_rn(__dadd_rn(ym, -__dmul_rn(2.0, y0)), yp);
        const double delta = denom != 0.0 ? __ddiv_rn(__dmul_rn(0.5, __dadd_rn(ym, -yp)), denom) : 0.0;
        s_pos[0] = (double)bs; s_pos[1] = delta;
        double* out = A.summary + (size_t)c * kNSummary;
        out[0] = (double)bs; out[1] = delta;
        out[2] = __ddiv_rn(__dadd_rn((double)bs, delta), A.f_s_hz);
        out[3] = y0; out[4] = s_sum[0];
    }
    __syncthreads();
    const uint32_t bs = (uint32_t)s_pos[0];
    const double delta = s_pos[1];

    // ---- group-delay corrected band-pass: B[i] = T[i] exp(+j 2 pi i (b* + delta) / N) ----
    for (uint32_t i = tid; i < N; i += kAnaThreads) {
        const uint32_t r = (uint32_t)(((uint64_t)i * bs) % N);
        const double turns = __dadd_rn(__ddiv_rn((double)r, (double)N), __ddiv_rn(__dmul_rn((double)i, delta), (double)N));
        double sn, cs;
        sincos(__dmul_rn(__dmul_rn(2.0, 3.14159265358979323846), turns), &sn, &cs);
        const double2 t = T[i];
        A.B[(size_t)c * N + i] = make_double2(t.x * cs - t.y * sn, t.x * sn + t.y * cs);
    }

    // ---- tone phases theta_i = arg T[i] + pi/2, in-band tones first .. K-1 ----
    const uint32_t K = N / 2, first = (A.zero_offset_mask >> c) & 1u;
    __syncthreads();                                  // power envelope no longer needed
    for (uint32_t i = first + tid; i < K; i += kAnaThreads) {
        const double2 t = T[i];
        ana_sm[i] = __dadd_rn(atan2(t.y, t.x), __dmul_rn(0.5, 3.14159265358979323846));
    }
    __syncthreads();
    if (tid != 0) return;
    // sequential unwrap + least squares (K <= 2048 terms; a few microseconds on one thread)
    const double two_pi = __dmul_rn(2.0, 3.14159265358979323846);
    double prev = 0.0, sx = 0.0, sy = 0.0, sxx = 0.0, sxy = 0.0;
    for (uint32_t i = first; i < K; ++i) {
        double th = ana_sm[i];
        if (i != first) {
            double d = __dadd_rn(th, -prev);
            d = __dadd_rn(d, -__dmul_rn(two_pi, floor(__dadd_rn(__ddiv_rn(d, two_pi), 0.5))));
            th = __dadd_rn(prev, d);
        }
        ana_sm[i] = th;
        prev = th;
        const double x = (double)i;
        sx += x; sy += th; sxx = __dadd_rn(sxx, __dmul_rn(x, x)); sxy = __dadd_rn(sxy, __dmul_rn(x, th));
    }
    const double n = (double)(K - first);
    const double det = __dadd_rn(__dmul_rn(n, sxx), -__dmul_rn(sx, sx));
    const double s = det != 0.0 ? __ddiv_rn(__dadd_rn(__dmul_rn(n, sxy), -__dmul_rn(sx, sy)), det) : 0.0;
    const double a = K > first ? __ddiv_rn(__dadd_rn(sy, -__dmul_rn(s, sx)), n) : 0.0;
    double rss = 0.0;
    for (uint32_t i = first; i < K; ++i) {
        const double r = __dadd_rn(ana_sm[i], -__dadd_rn(a, __dmul_rn(s, (double)i)));
        rss = __dadd_rn(rss, __dmul_rn(r, r));
    }
    double* out = A.summary + (size_t)c * kNSummary;
    out[5] = __ddiv_rn(s, __dmul_rn(two_pi, A.f_comb_hz));
    out[6] = a;
    out[7] = K > first ? sqrt(__ddiv_rn(rss, n)) : 0.0;
}

// ---- residual rotation of a time series of short integrations ----------------
// "... multiple passes over the x[n] input data, iteratively counter-rotating the input data
// using the residual phase shift detected in the previous pass."  Reading (R27): if eq. 2.3 rotates
// by f_rot while the comb sits at i f_comb + f_true, every tone phasor turns by 2 pi (f_true - f_rot) T_int
// from one short integration to the next, so
//     S = sum_{m < M-1} sum_{i in band} T_{m+1}[i] conj(T_m[i]),   residual phase shift = arg S.
// One CTA per channel; thread t adds the terms e = t, t + 256, ... (e = m * band + i, the oracle's order within
// a thread), then a fixed tree adds the 256 thread sums: deterministic.  out[c] = (arg S, |S|, sum |T_{m+1}||T_m|).
constexpr int kNResidual = 3;   // == PCAL_N_RESIDUAL
__global__ void __launch_bounds__(kAnaThreads) residual_rotation_kernel(const double2* __restrict__ T, uint32_t M, uint32_t N, uint32_t C,
                                                                        uint32_t zero_offset_mask, double* __restrict__ out) {
    __shared__ double s_re[kAnaThreads], s_im[kAnaThreads], s_nm[kAnaThreads];
    const uint32_t c = blockIdx.x, tid = threadIdx.x;
    const uint32_t i0 = (zero_offset_mask >> c) & 1u, band = N / 2 - i0;
    const uint32_t total = (M > 0 ? M - 1 : 0) * band;
    double re = 0.0, im = 0.0, nm = 0.0;
    for (uint32_t e = tid; e < total; e += kAnaThreads) {
        const uint32_t m = e / band, i = i0 + e % band;
        const double2 a = T[((size_t)(m + 1) * C + c) * N + i], b = T[((size_t)m * C + c) * N + i];
        re += a.x * b.x + a.y * b.y;
        im += a.y * b.x - a.x * b.y;
        nm += sqrt(a.x * a.x + a.y * a.y) * sqrt(b.x * b.x + b.y * b.y);
    }
    s_re[tid] = re; s_im[tid] = im; s_nm[tid] = nm;
    __syncthreads();
    for (uint32_t s = kAnaThreads / 2; s > 0; s >>= 1) {
        if (tid < s) { s_re[tid] += s_re[tid + s]; s_im[tid] += s_im[tid + s]; s_nm[tid] += s_nm[tid + s]; }
        __syncthreads();
    }
    if (tid == 0) {
        out[c * kNResidual + 0] = atan2(s_im[0], s_re[0]);
        out[c * kNResidual + 1] = hypot(s_re[0], s_im[0]);
        out[c * kNResidual + 2] = s_nm[0];
    }
}

}  // namespace pcal
