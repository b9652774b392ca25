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
#include "pcal_tail.cuh"

namespace pcal {

struct FoldParams {
    const uint4* data;      // [device] packed samples, 16-byte aligned
    uint64_t n_vec;         // complete 16-byte vectors in this launch
    uint32_t q;             // slot groups
    uint32_t R;             // replicas per slot group (gridDim.x == q*R)
    uint32_t n_iter;        // loop trips per warp (multiple of 16)
    uint32_t n_quot;        // n_vec / (threads in the grid): loads every thread makes ...
    uint64_t n_rem;         // ... plus one for the threads whose first vector index is < n_vec % threads
    void* partial;          // [device] per-CTA partial sums, layout [cta][field][lane]
    int input_ready;        // caller promised the input is complete: stream it before pdl_wait()
    TailParams tail;        // fused reduction + rotation by the CTAs that finish last (pcal_tail.cuh)
};

__device__ __forceinline__ uint64_t fold_first_vec(const FoldParams& P, int w, int lane) {
    const uint32_t p = blockIdx.x % P.q, rho0 = blockIdx.x / P.q;
    return ((uint64_t)(rho0 * kWarps + w) * P.q + p) * 32u + (uint32_t)lane;
}

// ---------------------------------------------------------------------------------------------
// 2-bit samples: 64 fields per vector.  Per-field sums of the (offset-binary) codes.
//
// The loads of one thread feed a streaming vertical counter (Harley-Seal): csa(plane, x0, x1)
// keeps the running plane of weight w and emits one carry word of weight 2w; 15 CSAs (30 LOP3)
// per word position turn 16 loads into the running planes O, T, F, E (weights 1, 2, 4, 8) and
// ONE word of weight 16, which alone is widened by SWAR (2-bit -> 4-bit lanes in registers,
// -> 16-bit lanes in shared memory every 5 groups).  About 0.15 integer instructions per
// sample, all exact.  Loads are software-pipelined: the next block of U 128-bit loads is issued
// before the current block is reduced, so every warp always has U..2U loads in flight.
// Output: uint16 partial[cta][64 fields][32 lanes], field f = bit pair 2f..2f+1 of the vector.
// Host guarantees n_iter <= 2048 (8 warps * 3 * n_iter < 65536) and n_iter % 16 == 0.
// ---------------------------------------------------------------------------------------------
constexpr int kFoldGroup = 16;   // loads per complete counter cascade

template <bool SIGN_MAG, int U, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) fold_2bit_kernel(const __grid_constant__ FoldParams P) {
    if (!P.input_ready) pdl_wait();
    static_assert(U == 4 || U == 8, "block of 4 or 8 loads");
    __shared__ uint32_t s_gen[3];
    __shared__ __align__(16) uint32_t hlf[32][kThreads];   // weight-16 sums in 16-bit lanes: [8j + f8] = fields f8, f8+8 of word j
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint64_t first = fold_first_vec(P, w, lane);
    const uint64_t stride = (uint64_t)P.R * kWarps * P.q * 32u;
    const uint32_t n_valid = P.n_quot + (first < P.n_rem ? 1u : 0u);   // this thread's real loads
    const uint4* base = P.data + first;
    // a vector that does not exist must add 0 to every code sum: raw pattern whose code is 0
    const uint32_t fill = SIGN_MAG ? 0xFFFFFFFFu : 0u;

#pragma unroll
    for (int h = 0; h < 32; ++h) hlf[h][tid] = 0;
    uint32_t O[4] = {0, 0, 0, 0}, T[4] = {0, 0, 0, 0}, F[4] = {0, 0, 0, 0}, E[4] = {0, 0, 0, 0};
    uint32_t nib[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // weight 16, 4-bit lanes: [2j+par] nibble i = field 2i+par
    uint32_t d[4], e[4];                             // pending carries of weight 4 and 8

    auto load_block = [&](uint4(&v)[U], uint32_t i0) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t i = i0 + u;
            v[u] = (i < n_valid) ? ldg_stream(base + (uint64_t)i * stride) : make_uint4(fill, fill, fill, fill);
        }
    };
    // four loads -> planes O, T updated, one carry word of weight 4 per word position
    auto quad = [&](const uint4& v0, const uint4& v1, const uint4& v2, const uint4& v3, uint32_t(&out4)[4]) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t x0 = word_of(v0, j), x1 = word_of(v1, j), x2 = word_of(v2, j), x3 = word_of(v3, j);
            if (SIGN_MAG) {
                x0 = signmag_to_offset_binary(x0); x1 = signmag_to_offset_binary(x1);
                x2 = signmag_to_offset_binary(x2); x3 = signmag_to_offset_binary(x3);
            }
            uint32_t ca, cb;
            csa(O[j], x0, x1, O[j], ca);
            csa(O[j], x2, x3, O[j], cb);
            csa(T[j], ca, cb, T[j], out4[j]);
        }
    };
    auto fold8 = [&](const uint32_t(&d0)[4], const uint32_t(&d1)[4], uint32_t(&out8)[4]) {
#pragma unroll
        for (int j = 0; j < 4; ++j) csa(F[j], d0[j], d1[j], F[j], out8[j]);
    };
    auto fold16 = [&](const uint32_t(&e0)[4], const uint32_t(&e1)[4]) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t g;
            csa(E[j], e0[j], e1[j], E[j], g);
            nib[2 * j] += g & 0x33333333u;
            nib[2 * j + 1] += (g >> 2) & 0x33333333u;
        }
    };
    auto flush_nib = [&]() {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int j = r >> 1, par = r & 1;
#pragma unroll
            for (int k = 0; k < 4; ++k) hlf[8 * j + 2 * k + par][tid] += (nib[r] >> (4 * k)) & 0x000F000Fu;
            nib[r] = 0;
        }
    };
    // one block of U loads; `phase` = index of the block inside its group of 16 loads
    auto reduce_block = [&](const uint4(&v)[U], int phase) {
        uint32_t d1[4], e1[4];
        if (U == 4) {
            if (phase == 0) quad(v[0], v[1], v[2], v[3], d);
            else if (phase == 1) { quad(v[0], v[1], v[2], v[3], d1); fold8(d, d1, e); }
            else if (phase == 2) quad(v[0], v[1], v[2], v[3], d);
            else { quad(v[0], v[1], v[2], v[3], d1); fold8(d, d1, e1); fold16(e, e1); }
        } else {
            quad(v[0], v[1], v[2], v[3], d);
            quad(v[4 % U], v[5 % U], v[6 % U], v[7 % U], d1);
            if (phase == 0) fold8(d, d1, e);
            else { fold8(d, d1, e1); fold16(e, e1); }
        }
    };

    uint4 bufA[U], bufB[U];
    load_block(bufA, 0);
    fold_ticket_and_release(P.tail, s_gen);   // first loads are in flight
    uint32_t groups_since_flush = 0;
    for (uint32_t i = 0; i < P.n_iter; i += kFoldGroup) {
#pragma unroll
        for (int b = 0; b < kFoldGroup / U; b += 2) {
            load_block(bufB, i + (b + 1) * U);
            reduce_block(bufA, b);
            load_block(bufA, i + (b + 2) * U);
            reduce_block(bufB, b + 1);
        }
        if (++groups_since_flush == 5) { flush_nib(); groups_since_flush = 0; }   // 4-bit lanes hold <= 15
    }
    flush_nib();

    // total = 16*hlf + val(O) + 2 val(T) + 4 val(F) + 8 val(E), assembled in 16-bit lanes
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const uint32_t m = 0x03030303u;   // byte i = field 4i + a
            const uint32_t v = ((O[j] >> (2 * a)) & m) + 2u * ((T[j] >> (2 * a)) & m) +
                               4u * ((F[j] >> (2 * a)) & m) + 8u * ((E[j] >> (2 * a)) & m);   // <= 45 per byte
            hlf[8 * j + a][tid] = 16u * hlf[8 * j + a][tid] + (v & 0x00FF00FFu);
            hlf[8 * j + a + 4][tid] = 16u * hlf[8 * j + a + 4][tid] + ((v >> 8) & 0x00FF00FFu);
        }
    }
    __syncthreads();
    fold_wait_slot(P.tail, s_gen);
    void* partial = fold_partial_of(P.tail, P.partial, s_gen);
    uint16_t* out = reinterpret_cast<uint16_t*>(partial) + (size_t)blockIdx.x * 64 * 32;
#pragma unroll
    for (int x = tid; x < 32 * 32; x += kThreads) {
        const int h = x >> 5, ln = x & 31;
        uint32_t s = 0;
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) s += hlf[h][ww * 32 + ln];  // 16-bit lanes, < 65536 by host cap
        const int f = 16 * (h >> 3) + (h & 7);
        out[f * 32 + ln] = (uint16_t)(s & 0xFFFFu);
        out[(f + 8) * 32 + ln] = (uint16_t)(s >> 16);
    }
    if (P.tail.enabled) fold_tail<KIND_2BIT>(P.tail, partial, P.q, P.R, reinterpret_cast<double*>(&hlf[0][0]), s_gen[0], s_gen[1]);
}

// ---------------------------------------------------------------------------------------------
// int8 samples: 16 fields per vector, exact int32 sums via DP4A with a one-hot byte selector.
// Output: int32 partial[cta][16][32].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, 3) fold_i8_kernel(const __grid_constant__ FoldParams P) {
    if (!P.input_ready) pdl_wait();
    __shared__ uint32_t s_gen[3];
    __shared__ __align__(16) int32_t sh[kWarps][16][32];   // also the (double) scratch of the fused tail
    fold_ticket_and_release(P.tail, s_gen);
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
    fold_wait_slot(P.tail, s_gen);
    void* partial = fold_partial_of(P.tail, P.partial, s_gen);
    int32_t* out = reinterpret_cast<int32_t*>(partial) + (size_t)blockIdx.x * 16 * 32;
    for (int e = threadIdx.x; e < 16 * 32; e += kThreads) {
        const int f = e >> 5, ln = e & 31;
        int32_t s = 0;
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) s += sh[ww][f][ln];
        out[f * 32 + ln] = s;
    }
    if (P.tail.enabled) fold_tail<KIND_I8>(P.tail, partial, P.q, P.R, reinterpret_cast<double*>(&sh[0][0][0]), s_gen[0], s_gen[1]);
}

// ---------------------------------------------------------------------------------------------
// float32 samples: 4 fields per vector.  Every sample is converted (exactly) and added in fp64: the folded bins of unrotated
// float32 input are REAL sums in which signal and noise cancel to a few per cent of a typical bin about once in a hundred
// bins, and fp32 runs of 16 additions (the first version: 1.7e-7 of a typical bin) put such bins outside 1e-5 relative.
// The price is two fp64-pipe instructions per sample (62 per clock and SM on B200): 0.4 us on a 16 MiB step
// (DESIGN.md "Accumulation precision").
// Output: double partial[cta][4][32].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, 3) fold_f32_kernel(const __grid_constant__ FoldParams P) {
    if (!P.input_ready) pdl_wait();
    __shared__ uint32_t s_gen[3];
    __shared__ __align__(16) double sh[kWarps][4][32];   // 1024 doubles: also the scratch of the fused tail
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint64_t idx = fold_first_vec(P, w, lane);
    const uint64_t stride = (uint64_t)P.R * kWarps * P.q * 32u;
    fold_ticket_and_release(P.tail, s_gen);
    double tot[4] = {0.0, 0.0, 0.0, 0.0};
    for (uint32_t i = 0; i < P.n_iter; i += kUnroll) {
        uint4 v[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const uint64_t a = idx + (uint64_t)u * stride;
            v[u] = (a < P.n_vec) ? ldg_stream(P.data + a) : make_uint4(0, 0, 0, 0);
        }
        idx += (uint64_t)kUnroll * stride;
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            tot[0] += (double)__uint_as_float(v[u].x);
            tot[1] += (double)__uint_as_float(v[u].y);
            tot[2] += (double)__uint_as_float(v[u].z);
            tot[3] += (double)__uint_as_float(v[u].w);
        }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) sh[w][k][lane] = tot[k];
    __syncthreads();
    fold_wait_slot(P.tail, s_gen);
    void* partial = fold_partial_of(P.tail, P.partial, s_gen);
    double* out = reinterpret_cast<double*>(partial) + (size_t)blockIdx.x * 4 * 32;
    for (int e = threadIdx.x; e < 4 * 32; e += kThreads) {
        const int f = e >> 5, ln = e & 31;
        double s = 0.0;
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) s += sh[ww][f][ln];  // fixed warp order: deterministic
        out[f * 32 + ln] = s;
    }
    if (P.tail.enabled) fold_tail<KIND_F32>(P.tail, partial, P.q, P.R, &sh[0][0][0], s_gen[0], s_gen[1]);
}

}  // namespace pcal
