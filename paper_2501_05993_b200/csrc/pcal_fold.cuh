// pcal_fold.cuh -- the hot kernels of the LUT / zero-offset path ("fold first, rotate once").
//
// eq. 2.3 + eq. 2.2 ask for P[b] = sum_n x[n] e^{-j w_off n} over n = b mod N_bins.
// When the rotator is periodic (eq. 2.4) the product only depends on n mod M for
// any M that is a multiple of L = lcm(N_bins, N_rotator), so
//     P[b] = sum_{r = b mod N_bins, r < M} e^{-j w_off r} * A[r],   A[r] = sum_{n = r mod M} x[n].
// This is the reordering the paper itself suggests ("accumulating into a
// N_rotator-sample accumulator and ... folding the long accumulator ... outside the samplecount
// loop").  The per-sample work becomes an integer add and is exact; the L complex MACs happen once
// per call in pcal_post.cuh.
//
// Thread/data mapping.  The input is a stream of 16-byte vectors; M is chosen as a multiple of the
// samples per vector, S = M / samples_per_vector "slots".  A warp load is 32 consecutive vectors
// (512 contiguous bytes).  Chunk kappa (32 vectors) starts at slot (32 kappa) mod S, which depends
// only on kappa mod q, q = S / gcd(S, 32).  CTA c owns slot group p = c mod q and replica
// rho0 = c / q; its warp w visits the chunks
//     kappa = ((rho0*8 + w) + i*R*8) * q + p,   i = 0, 1, ...          (R = gridDim.x / q)
// so every lane always lands on the same slot, i.e. on fixed residues mod M: its accumulators
// live in registers for the whole kernel, no atomics, no shared memory in the loop, and at every
// i the CTAs together read one contiguous range of the input (grid-stride, fully coalesced).
#pragma once
#include "pcal_common.cuh"

namespace pcal {

struct FoldParams {
    const uint4* data;      // [device] packed samples, 16-byte aligned
    uint64_t n_vec;         // complete 16-byte vectors in this launch
    uint32_t q;             // slot groups
    uint32_t R;             // replicas per slot group (gridDim.x == q*R)
    uint32_t n_iter;        // loop trips per warp (multiple of kUnroll)
    void* partial;          // [device] per-CTA partial sums, layout [cta][field][lane]
};

__device__ __forceinline__ uint64_t fold_first_vec(const FoldParams& P, int w, int lane) {
    const uint32_t p = blockIdx.x % P.q, rho0 = blockIdx.x / P.q;
    return ((uint64_t)(rho0 * kWarps + w) * P.q + p) * 32u + (uint32_t)lane;
}

// ---------------------------------------------------------------------------------------------
// 2-bit samples: 64 fields per vector.  Per-field sums of the (offset-binary) codes.
//
// Eight loads of one thread are compressed with a carry-save adder tree (7 CSAs = 14 LOP3 per
// word position) into running planes of weight 1, 2, 4 plus one word of weight 8 per group; only
// that word (one per 8 loads) goes through SWAR widening 2 -> 4 -> 8 -> 16 bits.  About 0.17
// integer instructions per sample, all exact.
// Output: uint16 partial[cta][64 fields][32 lanes], field f = bit pair 2f..2f+1 of the vector.
// Host guarantees n_iter <= 2048 so that 8 warps * 3 * n_iter < 65536.
// ---------------------------------------------------------------------------------------------
template <bool SIGN_MAG>
__global__ void __launch_bounds__(kThreads, 2) fold_2bit_kernel(FoldParams P) {
    __shared__ uint32_t sh[kWarps][32][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint64_t idx = fold_first_vec(P, w, lane);
    const uint64_t stride = (uint64_t)P.R * kWarps * P.q * 32u;
    // a vector that does not exist must add 0 to every code sum: raw pattern whose code is 0
    const uint32_t fill = SIGN_MAG ? 0xFFFFFFFFu : 0u;

    uint32_t ones[4] = {0, 0, 0, 0}, twos[4] = {0, 0, 0, 0}, fours[4] = {0, 0, 0, 0};
    uint32_t nib[8], byt[16], hlf[32];
#pragma unroll
    for (int k = 0; k < 8; ++k) nib[k] = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) byt[k] = 0;
#pragma unroll
    for (int k = 0; k < 32; ++k) hlf[k] = 0;

    uint32_t i = 0;
    while (i < P.n_iter) {
        for (int mid = 0; mid < 16 && i < P.n_iter; ++mid) {
            for (int inner = 0; inner < 5 && i < P.n_iter; ++inner, i += kUnroll) {
                uint4 v[kUnroll];
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) {
                    const uint64_t a = idx + (uint64_t)u * stride;
                    v[u] = (a < P.n_vec) ? ldg_stream(P.data + a) : make_uint4(fill, fill, fill, fill);
                }
                idx += (uint64_t)kUnroll * stride;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint32_t x[kUnroll];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) {
                        x[u] = word_of(v[u], j);
                        if (SIGN_MAG) x[u] = signmag_to_offset_binary(x[u]);
                    }
                    uint32_t s1, c1, s2, c2, s3, c3, s4, c4, t1, d1, t2, d2, f1, e1;
                    csa(x[0], x[1], x[2], s1, c1);
                    csa(x[3], x[4], x[5], s2, c2);
                    csa(s1, s2, x[6], s3, c3);
                    csa(s3, x[7], ones[j], s4, c4);
                    ones[j] = s4;
                    csa(c1, c2, c3, t1, d1);
                    csa(t1, c4, twos[j], t2, d2);
                    twos[j] = t2;
                    csa(d1, d2, fours[j], f1, e1);
                    fours[j] = f1;
                    // e1: fields of weight 8, values 0..3 -> 4-bit lanes (<= 5 additions)
                    nib[2 * j] += e1 & 0x33333333u;
                    nib[2 * j + 1] += (e1 >> 2) & 0x33333333u;
                }
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {  // 4-bit -> 8-bit lanes (<= 16*15 = 240)
                byt[2 * k] += nib[k] & 0x0F0F0F0Fu;
                byt[2 * k + 1] += (nib[k] >> 4) & 0x0F0F0F0Fu;
                nib[k] = 0;
            }
        }
#pragma unroll
        for (int k = 0; k < 16; ++k) {  // 8-bit -> 16-bit lanes
            hlf[2 * k] += byt[k] & 0x00FF00FFu;
            hlf[2 * k + 1] += (byt[k] >> 8) & 0x00FF00FFu;
            byt[k] = 0;
        }
    }

    // total = 8*hlf + 4*val(fours) + 2*val(twos) + val(ones), all in the 16-bit lane layout:
    // register h = ((2j + par)*2 + hi4)*2 + hi8 holds fields 16j + a + 4*hi8 (+8 in the upper
    // half-word), a = par + 2*hi4.
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int par = 0; par < 2; ++par) {
            const uint32_t m3 = 0x33333333u;
            const uint32_t n1 = (par ? (ones[j] >> 2) : ones[j]) & m3;
            const uint32_t n2 = (par ? (twos[j] >> 2) : twos[j]) & m3;
            const uint32_t n4 = (par ? (fours[j] >> 2) : fours[j]) & m3;
#pragma unroll
            for (int hi4 = 0; hi4 < 2; ++hi4) {
                const uint32_t b1 = (hi4 ? (n1 >> 4) : n1) & 0x0F0F0F0Fu;
                const uint32_t b2 = (hi4 ? (n2 >> 4) : n2) & 0x0F0F0F0Fu;
                const uint32_t b4 = (hi4 ? (n4 >> 4) : n4) & 0x0F0F0F0Fu;
                const uint32_t bs = b1 + 2u * b2 + 4u * b4;  // <= 21 per byte
#pragma unroll
                for (int hi8 = 0; hi8 < 2; ++hi8) {
                    const int h = ((2 * j + par) * 2 + hi4) * 2 + hi8;
                    hlf[h] = 8u * hlf[h] + ((hi8 ? (bs >> 8) : bs) & 0x00FF00FFu);
                }
            }
        }
    }
#pragma unroll
    for (int h = 0; h < 32; ++h) sh[w][h][lane] = hlf[h];
    __syncthreads();
    uint16_t* out = reinterpret_cast<uint16_t*>(P.partial) + (size_t)blockIdx.x * 64 * 32;
#pragma unroll
    for (int e = threadIdx.x; e < 32 * 32; e += kThreads) {
        const int h = e >> 5, ln = e & 31;
        uint32_t s = 0;
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) s += sh[ww][h][ln];  // 16-bit lanes, < 65536 by host cap
        const int hi8 = h & 1, hi4 = (h >> 1) & 1, par = (h >> 2) & 1, j = h >> 3;
        const int f = 16 * j + par + 2 * hi4 + 4 * hi8;
        out[f * 32 + ln] = (uint16_t)(s & 0xFFFFu);
        out[(f + 8) * 32 + ln] = (uint16_t)(s >> 16);
    }
}

// ---------------------------------------------------------------------------------------------
// int8 samples: 16 fields per vector, exact int32 sums via DP4A with a one-hot byte selector.
// Output: int32 partial[cta][16][32].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, 3) fold_i8_kernel(FoldParams P) {
    __shared__ int32_t sh[kWarps][16][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint64_t idx = fold_first_vec(P, w, lane);
    const uint64_t stride = (uint64_t)P.R * kWarps * P.q * 32u;
    int32_t acc[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = 0;
    for (uint32_t i = 0; i < P.n_iter; i += kUnroll) {
        uint4 v[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const uint64_t a = idx + (uint64_t)u * stride;
            v[u] = (a < P.n_vec) ? ldg_stream(P.data + a) : make_uint4(0, 0, 0, 0);
        }
        idx += (uint64_t)kUnroll * stride;
#pragma unroll
        for (int u = 0; u < kUnroll; ++u)
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    acc[4 * j + k] = __dp4a((int)word_of(v[u], j), 1 << (8 * k), acc[4 * j + k]);
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) sh[w][k][lane] = acc[k];
    __syncthreads();
    int32_t* out = reinterpret_cast<int32_t*>(P.partial) + (size_t)blockIdx.x * 16 * 32;
    for (int e = threadIdx.x; e < 16 * 32; e += kThreads) {
        const int f = e >> 5, ln = e & 31;
        int32_t s = 0;
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) s += sh[ww][f][ln];
        out[f * 32 + ln] = s;
    }
}

// ---------------------------------------------------------------------------------------------
// float32 samples: 4 fields per vector.  fp32 runs of 16 additions, flushed into fp64
// (runs <= 64 keep every bin within 1.3e-6 relative).
// Output: double partial[cta][4][32].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, 3) fold_f32_kernel(FoldParams P) {
    __shared__ double sh[kWarps][4][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint64_t idx = fold_first_vec(P, w, lane);
    const uint64_t stride = (uint64_t)P.R * kWarps * P.q * 32u;
    double tot[4] = {0.0, 0.0, 0.0, 0.0};
    for (uint32_t i = 0; i < P.n_iter; i += 2 * kUnroll) {
        float run[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            uint4 v[kUnroll];
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                const uint64_t a = idx + (uint64_t)u * stride;
                v[u] = (a < P.n_vec) ? ldg_stream(P.data + a) : make_uint4(0, 0, 0, 0);
            }
            idx += (uint64_t)kUnroll * stride;
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                run[0] += __uint_as_float(v[u].x);
                run[1] += __uint_as_float(v[u].y);
                run[2] += __uint_as_float(v[u].z);
                run[3] += __uint_as_float(v[u].w);
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) tot[k] += (double)run[k];
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) sh[w][k][lane] = tot[k];
    __syncthreads();
    double* out = reinterpret_cast<double*>(P.partial) + (size_t)blockIdx.x * 4 * 32;
    for (int e = threadIdx.x; e < 4 * 32; e += kThreads) {
        const int f = e >> 5, ln = e & 31;
        double s = 0.0;
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) s += sh[ww][f][ln];  // fixed warp order: deterministic
        out[f * 32 + ln] = s;
    }
}

}  // namespace pcal
