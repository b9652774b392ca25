// pcal_post.cuh -- the small deterministic kernels behind the hot loop:
//   reduce_replicas_kernel   per-CTA partials -> one accumulator per (slot group, field, lane)
//                            (the "binary tree stepping" the paper leaves to the host)
//   rotate_fold_kernel       A[r] * exp(-j w_off r) folded to N_bins (eq. 2.3 + 2.2 after the
//                            reordering of PAPER.md:200), plus the ragged tail (< 1 vector)
//   gen_reduce_kernel        per-CTA generator partials -> bins
//   dft_kernel               T[i] = sum_b P[b] exp(-j 2 pi i b / N_bins)
// All sums run in a fixed order (no atomics): two runs give bit-identical results.
#pragma once
#include "pcal_common.cuh"

namespace pcal {

constexpr int kPostThreads = 128;

// ---- stage 1: sum the R replicas of each slot group -------------------------------------------
// in : T partial[(rho0*q + p)][F][32]      out: int64/double acc[p][F][32]
template <typename Tin, typename Tacc>
__global__ void reduce_replicas_kernel(const Tin* __restrict__ partial, Tacc* __restrict__ acc,
                                       uint32_t q, uint32_t R, uint32_t F) {
    const uint32_t per_group = F * 32u;
    const uint32_t total = q * per_group;
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= total) return;
    Tacc s = 0;
    for (uint32_t r = 0; r < R; ++r) s += (Tacc)partial[(size_t)r * total + x];  // fixed order
    acc[x] = s;
}

struct RotateParams {
    const void* acc;          // [device] int64 or double acc[q][F][32]
    const double2* lut;       // [device] concatenated per-channel rotator tables (eq. 2.4)
    const uint32_t* lut_off;  // [device] per channel: first entry
    const uint32_t* lut_len;  // [device] per channel: L_c (1 => no rotation)
    double2* P;               // [device] folded bins [C][N_bins], accumulated into
    long long* Pint;          // [device] exact integer bins [C][N_bins] (valid when no rotation)
    const uint8_t* tail;      // [device] first byte after the last complete vector
    uint64_t n0;              // absolute index of the first sample of this call
    uint64_t NT;              // time samples covered by complete vectors
    uint64_t n_total;         // time samples in this call
    uint32_t q, F, C;         // slot groups, fields per vector, channels
    uint32_t spv;             // time samples per vector
    uint32_t n_bins;
    int kind;                 // KIND_*
    int sign_mag;
    int integer_exact;        // also accumulate Pint
};

// decode one tail sample (time index t relative to the first tail byte's first sample)
__device__ __forceinline__ double tail_value(const RotateParams& P, uint32_t t, uint32_t c) {
    if (P.kind == KIND_F32) return (double)reinterpret_cast<const float*>(P.tail)[t];
    if (P.kind == KIND_I8) return (double)reinterpret_cast<const int8_t*>(P.tail)[t];
    const uint32_t bit = (t * P.C + c) * 2u;
    const uint32_t code = (P.tail[bit >> 3] >> (bit & 7u)) & 3u;
    if (P.sign_mag) return (code & 2u) ? -(double)(1 + 2 * (code & 1u)) : (double)(1 + 2 * (code & 1u));
    return (double)(2 * (int)code - 3);
}

// ---- stage 2: one block per (channel, bin) ---------------------------------------------------
// The super-row (q*32 vectors = SR time samples, a multiple of M and of N_bins) is the index space
// of acc: offset o in [0, SR) <-> (p, lane, time-in-vector).  Bin b collects the offsets
// o = o_b + j*N_bins.  For 2-bit data acc holds code sums; level sum = 2*acc - 3*count(o).
__global__ void __launch_bounds__(kPostThreads) rotate_fold_kernel(RotateParams P) {
    __shared__ double sre[kPostThreads], sim[kPostThreads];
    __shared__ long long sint[kPostThreads];
    const uint32_t c = blockIdx.y, b = blockIdx.x;
    const uint64_t SR = (uint64_t)P.q * 32u * P.spv;
    const uint32_t L = P.lut_len[c];
    const double2* lut = P.lut + P.lut_off[c];
    const uint32_t o_b = (uint32_t)(((uint64_t)b + P.n_bins - (P.n0 % P.n_bins)) % P.n_bins);
    const uint32_t n0L = (uint32_t)(P.n0 % L);
    double are = 0.0, aim = 0.0;
    long long aint = 0;
    for (uint64_t o = o_b + (uint64_t)threadIdx.x * P.n_bins; o < SR; o += (uint64_t)kPostThreads * P.n_bins) {
        if (o >= P.NT) break;
        const uint32_t vec = (uint32_t)(o / P.spv), tf = (uint32_t)(o % P.spv);
        const uint32_t p = vec >> 5, lane = vec & 31u;
        const uint32_t f = tf * P.C + c;
        const size_t x = ((size_t)p * P.F + f) * 32u + lane;
        double val;
        long long ival = 0;
        if (P.kind == KIND_F32) {
            val = reinterpret_cast<const double*>(P.acc)[x];
        } else {
            ival = reinterpret_cast<const long long*>(P.acc)[x];
            if (P.kind == KIND_2BIT) {
                const long long cnt = (long long)((P.NT - o - 1) / SR + 1);
                ival = 2 * ival - 3 * cnt;
            }
            val = (double)ival;
        }
        if (L > 1) {
            const double2 ph = lut[(n0L + (uint32_t)(o % L)) % L];
            are += val * ph.x;
            aim += val * ph.y;
        } else {
            are += val;
            aint += ival;
        }
    }
    sre[threadIdx.x] = are; sim[threadIdx.x] = aim; sint[threadIdx.x] = aint;
    __syncthreads();
    for (int s = kPostThreads / 2; s > 0; s >>= 1) {  // fixed tree
        if (threadIdx.x < s) {
            sre[threadIdx.x] += sre[threadIdx.x + s];
            sim[threadIdx.x] += sim[threadIdx.x + s];
            sint[threadIdx.x] += sint[threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double tre = sre[0], tim = sim[0];
        long long tint = sint[0];
        // ragged tail: samples NT .. n_total-1 (fewer than one vector)
        for (uint64_t t = P.NT; t < P.n_total; ++t) {
            if ((P.n0 + t) % P.n_bins != b) continue;
            const double v = tail_value(P, (uint32_t)(t - P.NT), c);
            if (L > 1) {
                const double2 ph = lut[(n0L + (uint32_t)(t % L)) % L];
                tre += v * ph.x; tim += v * ph.y;
            } else {
                tre += v; tint += (long long)v;
            }
        }
        double2 cur = P.P[(size_t)c * P.n_bins + b];
        cur.x += tre; cur.y += tim;
        P.P[(size_t)c * P.n_bins + b] = cur;
        if (P.integer_exact) P.Pint[(size_t)c * P.n_bins + b] += tint;
    }
}

// ---- DFT of the folded period ------------------------------------------------------------------
// T[c][i] = sum_b P[c][b] * W[(i'*b) mod N], i' = (i - k_shift) mod N, W[k] = exp(-j 2 pi k/N)
// (twiddle table built on the host in long double).  One thread per output, fixed order in b.
__global__ void dft_kernel(const double2* __restrict__ P, const double2* __restrict__ W,
                           double2* __restrict__ T, uint32_t N, uint32_t k_shift) {
    extern __shared__ double2 sm[];  // [N] bins of this channel, [N] twiddles
    double2* sp = sm;
    double2* sw = sm + N;
    const uint32_t c = blockIdx.y;
    for (uint32_t t = threadIdx.x; t < N; t += blockDim.x) {
        sp[t] = P[(size_t)c * N + t];
        sw[t] = W[t];
    }
    __syncthreads();
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t ii = (i + N - k_shift % N) % N;
    double re = 0.0, im = 0.0;
    uint32_t k = 0;
    for (uint32_t b = 0; b < N; ++b) {
        const double2 p = sp[b], w = sw[k];
        re += p.x * w.x - p.y * w.y;
        im += p.x * w.y + p.y * w.x;
        k += ii; if (k >= N) k -= N;
    }
    T[(size_t)c * N + i] = make_double2(re, im);
}

__global__ void zero_kernel(double2* P, long long* Pint, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { P[i] = make_double2(0.0, 0.0); Pint[i] = 0; }
}

__global__ void add_bins_kernel(double2* P, const double2* add, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { P[i].x += add[i].x; P[i].y += add[i].y; }
}

}  // namespace pcal
