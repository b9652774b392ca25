// pcal_gen.cuh -- the hot kernel of the sinewave-generator path (eq. 2.5-2.9).
//
// Needed when the rotator period is impractical ("prime valued frequency
// offsets"), e.g. BASELINE.json config 5 (f_offset = 1234.567 Hz), and runnable on any
// single-channel input (config 3, generator variant).
//
// What is kept from the paper: a recursive fixed-frequency oscillator advanced by a constant
// phase increment (eq. 2.5) instead of a table; the coupled form (eq. 2.6, a plain complex
// multiply by e^{-j dphi}) is used because its error does not blow up for small dphi the way the
// DFR does; stride-S stepping (eq. 2.8: "2cos(2 dphi)") is generalised to S = one
// CTA iteration.  What is different on a B200: one oscillator per THREAD, stepped once per
// 16-byte/4-byte load instead of once per sample, because
//     sum_q x[n_q + k] e^{-j w (n_q + k)} = e^{-j w k} * sum_q x[n_q + k] e^{-j w n_q}
// (the same algebra as the paper's k-shift): all SPT samples of a load share ONE
// phasor and the constant e^{-j w k} is applied once at the end.  Oscillator state is fp64; at
// the start of every 2^16-sample tile it is re-derived from the exactly reduced INTEGER phase
// (n * F_off) mod F_s -- BASELINE.json config 5's "fp64 phase resync every 2^16 samples".
//
// Mapping: a CTA iteration covers `span` consecutive samples (thread t owns samples
// t*SPT .. t*SPT+SPT-1 of it; span = a multiple of lcm(N_bins, SPT), so every thread keeps fixed
// bins).  gen_kernel: the piece's iterations are split into gridDim.x equal contiguous ranges (a
// short piece still loads every SM alike), a range is walked in tiles of 65536/(kThreads*SPT)
// iterations, the last one partial.  gen_mma_kernel: whole tiles dealt round-robin to CTAs.
// Per-sample work: decode (2 integer ops) + one packed FFMA2 issue (re and im of two samples).
// fp32 partial sums live for one tile (<= 64 additions), then are added to fp64 accumulators in
// shared memory.
#pragma once
#include <type_traits>
#include "pcal_common.cuh"
#include "pcal_gen_tail.cuh"

namespace pcal {

constexpr uint32_t kTileSamples = 1u << 16;

struct GenParams {
    const void* data;        // [device] packed samples
    uint64_t n_loads;        // complete per-thread loads available (vectors of SPT samples)
    uint64_t n_tiles;        // gen_mma_kernel: tiles in the piece
    uint64_t n_iters;        // gen_kernel: CTA iterations in the piece (the last one may be partial)
    uint32_t span;           // samples per CTA iteration: the largest multiple of lcm(N_bins, SPT) <= kThreads*SPT (threads past it idle)
    uint64_t Fs, k0, E, D;   // micro-hertz sample rate; (n0*Foff)%Fs; (tile*Foff)%Fs; (grid*E)%Fs
    uint64_t Foff;
    double2 rho;             // exp(-j w * kThreads*SPT): oscillator step per CTA iteration
    double2 rho2;            // rho^2 (from the exactly reduced phase of two steps)
    double2 tw[16];          // exp(-j w k), k = 0..15: post-twiddle within a load
    GenTailParams tail;      // reduction, ragged tail, accumulation (and DFT) by the CTA that finishes last (pcal_gen_tail.cuh)
    uint32_t n_bins;
    int sign_mag;
    int input_ready;              // caller promised the input is complete: stream it before pdl_wait()
    uint32_t dec_mask, dec_one;   // 0x00600000, 0x3F800000 (2-bit decode, see lop3_and_or)
};

__device__ __forceinline__ void ffma2(float2& acc, const float2 x, const float2 c) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;"
        : "+l"(*reinterpret_cast<unsigned long long*>(&acc))
        : "l"(*reinterpret_cast<const unsigned long long*>(&x)),
          "l"(*reinterpret_cast<const unsigned long long*>(&c)));
}
__device__ __forceinline__ float2 fadd2(const float2 a, const float2 b) {
    float2 r;
    asm("add.rn.f32x2 %0, %1, %2;"
        : "=l"(*reinterpret_cast<unsigned long long*>(&r))
        : "l"(*reinterpret_cast<const unsigned long long*>(&a)),
          "l"(*reinterpret_cast<const unsigned long long*>(&b)));
    return r;
}

template <int KIND> struct GenTraits;
template <> struct GenTraits<KIND_F32>  { static constexpr int SPT = 4;  using Vec = uint4; };
template <> struct GenTraits<KIND_I8>   { static constexpr int SPT = 16; using Vec = uint4; };
template <> struct GenTraits<KIND_2BIT> { static constexpr int SPT = 16; using Vec = uint32_t; };

// decode one load into SPT floats.  2-bit: returns u = 1 + c/4 (c = offset-binary code), the
// caller undoes level = 8u - 11 in fp64 at the end; int8 / float32: the sample value itself.
template <int KIND>
__device__ __forceinline__ void gen_decode(const typename GenTraits<KIND>::Vec& v, float* x, int sign_mag);

template <>
__device__ __forceinline__ void gen_decode<KIND_F32>(const uint4& v, float* x, int) {
    x[0] = __uint_as_float(v.x); x[1] = __uint_as_float(v.y);
    x[2] = __uint_as_float(v.z); x[3] = __uint_as_float(v.w);
}
template <>
__device__ __forceinline__ void gen_decode<KIND_I8>(const uint4& v, float* x, int) {
    // byte b (two's complement) -> u = b ^ 0x80 in [0,255] -> float bits 0x4B0000uu = 2^23 + u
    // -> subtract 2^23 + 128: exact, no I2F conversion pipe.
    const float2 bias = make_float2(-8388736.0f, -8388736.0f);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t w = word_of(v, j) ^ 0x80808080u;
#pragma unroll
        for (int k = 0; k < 4; k += 2) {
            float2 p = make_float2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7440 | k)),
                                   __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7440 | (k + 1))));
            p = fadd2(p, bias);
            x[4 * j + k] = p.x; x[4 * j + k + 1] = p.y;
        }
    }
}
// (a & b) | c in ONE LOP3.  b and c are the decode constants 0x00600000 / 0x3F800000 handed over
// as kernel parameters (GenParams::dec_mask / dec_one): with immediates ptxas needs two LOP3,
// because one instruction can encode only one immediate.
__device__ __forceinline__ uint32_t lop3_and_or(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ void gen_decode_2bit(uint32_t v, float* x, int sign_mag, uint32_t dec_mask, uint32_t dec_one) {
    const uint32_t w = sign_mag ? signmag_to_offset_binary(v) : v;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const uint32_t sh = (2 * k <= 21) ? (w << (21 - 2 * k)) : (w >> (2 * k - 21));
        x[k] = __uint_as_float(lop3_and_or(sh, dec_mask, dec_one));  // 1 + c/4
    }
    // centre the code: (1 + c/4) - 1.375 = level/8 exactly.  Without it every fp32 sum would carry a
    // DC term ~ sum of phasors, whose rounding (not the signal's) would set the error floor.
    const float2 bias = make_float2(-1.375f, -1.375f);
#pragma unroll
    for (int k = 0; k < 16; k += 2) {
        const float2 p = fadd2(make_float2(x[k], x[k + 1]), bias);
        x[k] = p.x; x[k + 1] = p.y;
    }
}

// ---- own-thread asynchronous copies: global -> this thread's slot of a shared-memory ring ----
// Every thread prefetches ITS OWN future loads (cp.async), so completion is tracked per thread with
// cp.async.wait_group and no barrier is needed; the bytes in flight per SM (DEPTH loads per thread)
// do not cost registers.
template <int BYTES>
__device__ __forceinline__ void cp_async_own(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    static_assert(BYTES == 16 || BYTES == 8 || BYTES == 4, "cp.async sizes");
    if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
    else if (BYTES == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int kGenMaxTiles = 256;   // tiles per CTA per launch (host splits longer segments)

template <int KIND> struct GenCfg;
// LPT loads per thread per 2^16-sample tile; RUN tiles between fp32 -> fp64 flushes (<= 64 additions,
// the 2-bit code is centred to level/8 at decode, so its sums carry no DC term); DEPTH loads in flight per thread.
template <> struct GenCfg<KIND_F32>  { static constexpr int LB = 16, LPT = 64, RUN = 1, DEPTH = 16; };
template <> struct GenCfg<KIND_I8>   { static constexpr int LB = 16, LPT = 16, RUN = 4, DEPTH = 8; };
template <> struct GenCfg<KIND_2BIT> { static constexpr int LB = 4,  LPT = 16, RUN = 4, DEPTH = 16; };

template <int KIND>
constexpr size_t gen_smem_bytes() {
    return (size_t)GenTraits<KIND>::SPT * kThreads * sizeof(double2) + (size_t)kGenMaxTiles * sizeof(double2) +
           (size_t)GenCfg<KIND>::DEPTH * kThreads * GenCfg<KIND>::LB;
}

template <int KIND>
__global__ void __launch_bounds__(kThreads, 2) gen_kernel(const __grid_constant__ GenParams P) {
    if (!P.input_ready) pdl_wait();
    __shared__ uint32_t s_gen[4];
    constexpr int SPT = GenTraits<KIND>::SPT;
    constexpr int LB = GenCfg<KIND>::LB, LPT = GenCfg<KIND>::LPT, RUN = GenCfg<KIND>::RUN, DEPTH = GenCfg<KIND>::DEPTH;
    constexpr uint32_t SPAN = kThreads * SPT;                // samples per CTA iteration at most (a tile: LPT iterations, <= 2^16 samples)
    static_assert((uint32_t)LPT * SPAN == kTileSamples, "a full tile is 2^16 samples");
    const bool active = (uint32_t)threadIdx.x * SPT < P.span;   // N_bins that do not divide SPAN: the last threads have no samples
    using Vec = typename GenTraits<KIND>::Vec;
    extern __shared__ __align__(16) unsigned char gen_smem[];
    double2* acc = reinterpret_cast<double2*>(gen_smem);                 // [SPT][kThreads] (re, im)
    double2* base = acc + SPT * kThreads;                                 // [kGenMaxTiles] tile-start phasors
    unsigned char* ring = reinterpret_cast<unsigned char*>(base + kGenMaxTiles);   // [DEPTH][kThreads][LB]
    const int tid = threadIdx.x;
    const uint32_t dec_mask = P.dec_mask, dec_one = P.dec_one;   // opaque to ptxas: see lop3_and_or
#pragma unroll
    for (int k = 0; k < SPT; ++k) acc[k * kThreads + tid] = make_double2(0.0, 0.0);

    // this CTA's iterations: an equal share [it_lo, it_hi) of the piece, walked in tiles of LPT iterations
    const uint64_t it_lo = P.n_iters * blockIdx.x / gridDim.x, it_hi = P.n_iters * (blockIdx.x + 1ull) / gridDim.x;
    const uint32_t nt = (uint32_t)((it_hi - it_lo + LPT - 1) / LPT);
    const unsigned char* gdata = reinterpret_cast<const unsigned char*>(P.data);
    unsigned char* my_ring = ring + (size_t)tid * LB;
    constexpr size_t RING_STRIDE = (size_t)kThreads * LB;                // bytes between a thread's ring slots
    static_assert(LPT % DEPTH == 0, "ring slot of load j is j % DEPTH, a compile-time constant");
    const uint64_t LOAD_STRIDE = (uint64_t)(P.span / SPT) * LB;          // bytes between a thread's loads
    const uint64_t TILE_BYTES = (uint64_t)LPT * LOAD_STRIDE;
    const uint64_t end_off = it_hi * LOAD_STRIDE < P.n_loads * LB ? it_hi * LOAD_STRIDE : P.n_loads * LB;   // first byte past this CTA's last load
    const uint64_t tile_stride = TILE_BYTES;
    uint64_t off = it_lo * LOAD_STRIDE + (uint64_t)tid * LB;              // this thread's load 0 of tile i

    float2 ar[SPT / 2], ai[SPT / 2];
#pragma unroll
    for (int k2 = 0; k2 < SPT / 2; ++k2) { ar[k2] = make_float2(0.f, 0.f); ai[k2] = make_float2(0.f, 0.f); }

    static_assert(DEPTH % 2 == 0 && LPT % 2 == 0, "loads are committed and consumed in pairs");
#pragma unroll
    for (int j = 0; j < DEPTH; ++j) {                        // prologue: the first DEPTH loads of tile 0
        if (active && nt > 0 && off + j * LOAD_STRIDE < end_off)
            cp_async_own<LB>(my_ring + (size_t)j * RING_STRIDE, gdata + off + j * LOAD_STRIDE);
        if (j & 1) cp_async_commit();                        // one commit group per pair of loads
    }
    // (the first loads are in flight: now the ticket and the tables)
    if (tid == kThreads - 1) { if (P.tail.st) gen_take_ticket(P.tail, s_gen); }      // (published by the barrier below)
    // ---- resync table: the exactly reduced INTEGER phase of every tile start -> fp64 phasor ----
    for (uint32_t i = tid; i < nt; i += kThreads) {       // (k0 = phase of the piece's first sample)
        uint64_t k = P.k0 + mulmod_u64(P.Foff, (it_lo + (uint64_t)i * LPT) * P.span % P.Fs, P.Fs);
        if (k >= P.Fs) k -= P.Fs;
        base[i] = phasor_neg(k, P.Fs);
    }
    const double2 theta = phasor_neg(mulmod_u64(P.Foff, (uint64_t)tid * SPT, P.Fs), P.Fs);   // exp(-j w tid SPT)
    __syncthreads();
    pdl_release();            // the ticket is taken: the next launch may become resident

    const float rho_c = (float)P.rho.x, rho_s = (float)P.rho.y;

    // one tile; CHECK = false when this tile and the next one are complete (no per-load tests).
    // Loads are consumed in pairs: one wait, two ring reads, two refills, one commit.  The fp64
    // oscillator advances by rho^2 per pair; the second load's phasor is the first one turned by rho
    // in fp32 (one step, ~1e-7, never fed back into the fp64 state).
    auto tile_body = [&](auto check_tag, double2 ph, bool next_exists) {
        constexpr bool CHECK = decltype(check_tag)::value;
        auto mac = [&](const Vec& v, float c, float sn) {
            float x[SPT];
            if constexpr (KIND == KIND_2BIT) gen_decode_2bit(v, x, P.sign_mag, dec_mask, dec_one);
            else gen_decode<KIND>(v, x, P.sign_mag);
            const float2 cc = make_float2(c, c), ss = make_float2(sn, sn);
#pragma unroll
            for (int k2 = 0; k2 < SPT / 2; ++k2) {
                const float2 xx = make_float2(x[2 * k2], x[2 * k2 + 1]);
                ffma2(ar[k2], xx, cc);
                ffma2(ai[k2], xx, ss);
            }
        };
        auto refill = [&](int j, int slot) {                 // load j + DEPTH: same tile or the next one
            const uint64_t o = (j + DEPTH < LPT) ? off + (uint64_t)(j + DEPTH) * LOAD_STRIDE
                                                 : off + tile_stride + (uint64_t)(j + DEPTH - LPT) * LOAD_STRIDE;
            bool go = true;
            if (CHECK) go = ((j + DEPTH < LPT) || next_exists) && o < end_off;
            if (go && active) cp_async_own<LB>(my_ring + (size_t)slot * RING_STRIDE, gdata + o);
        };
#pragma unroll
        for (int j = 0; j < LPT; j += 2) {
            const int s0 = j % DEPTH, s1 = (j + 1) % DEPTH;  // compile-time after unrolling
            cp_async_wait<DEPTH / 2 - 1>();
            const Vec v0 = *reinterpret_cast<const Vec*>(my_ring + (size_t)s0 * RING_STRIDE);
            const Vec v1 = *reinterpret_cast<const Vec*>(my_ring + (size_t)s1 * RING_STRIDE);
            const float c0 = (float)ph.x, sn0 = (float)ph.y;
            const float c1 = __fmaf_rn(c0, rho_c, -sn0 * rho_s), sn1 = __fmaf_rn(c0, rho_s, sn0 * rho_c);
            bool ok0 = true, ok1 = true;
            if (CHECK) { ok0 = off + j * LOAD_STRIDE < end_off; ok1 = off + (j + 1) * LOAD_STRIDE < end_off; }
            if (ok0 && active) mac(v0, c0, sn0);
            if (ok1 && active) mac(v1, c1, sn1);
            refill(j, s0);
            refill(j + 1, s1);
            cp_async_commit();
            // coupled-form oscillator step (eq. 2.6) over two loads: ph *= rho^2, fp64
            const double nx = ph.x * P.rho2.x - ph.y * P.rho2.y;
            const double ny = ph.x * P.rho2.y + ph.y * P.rho2.x;
            ph.x = nx; ph.y = ny;
        }
    };

    for (uint32_t i = 0; i < nt; ++i, off += tile_stride) {
        // oscillator re-seeded at the tile start: exact tile phase x this thread's offset phasor
        const double2 b = base[i];
        const double2 ph0 = make_double2(b.x * theta.x - b.y * theta.y, b.x * theta.y + b.y * theta.x);
        const uint64_t tile0 = off - (uint64_t)tid * LB;     // first byte of tile i
        const bool next_exists = i + 1 < nt;
        const bool fast = tile0 + TILE_BYTES + (uint64_t)DEPTH * LOAD_STRIDE <= end_off;   // tile i and the first DEPTH iterations of tile i+1 complete
        if (fast) tile_body(std::false_type{}, ph0, true);
        else tile_body(std::true_type{}, ph0, next_exists);
        if ((i + 1) % RUN == 0 || i + 1 == nt) {
            // ---- flush the fp32 sums (<= 64 additions each) into the fp64 accumulators ----
#pragma unroll
            for (int k2 = 0; k2 < SPT / 2; ++k2) {
                double2 a0 = acc[(2 * k2) * kThreads + tid], a1 = acc[(2 * k2 + 1) * kThreads + tid];
                a0.x += (double)ar[k2].x; a0.y += (double)ai[k2].x;
                a1.x += (double)ar[k2].y; a1.y += (double)ai[k2].y;
                acc[(2 * k2) * kThreads + tid] = a0; acc[(2 * k2 + 1) * kThreads + tid] = a1;
                ar[k2] = make_float2(0.f, 0.f); ai[k2] = make_float2(0.f, 0.f);
            }
        }
    }
    cp_async_wait<0>();

    // ---- post-twiddle by exp(-j w k), undo the 2-bit affine code, reduce positions to bins ----
    double zr[SPT], zi[SPT];
#pragma unroll
    for (int k = 0; k < SPT; ++k) {
        const double2 a = acc[k * kThreads + tid];
        double re = a.x, im = a.y;
        if (KIND == KIND_2BIT) { re *= 8.0; im *= 8.0; }      // sums of level/8
        zr[k] = re * P.tw[k].x - im * P.tw[k].y;
        zi[k] = re * P.tw[k].y + im * P.tw[k].x;
    }
    __syncthreads();
    double* pos_re = reinterpret_cast<double*>(gen_smem);   // [SPAN]
    double* pos_im = pos_re + SPAN;                           // [SPAN]   (together == the acc region)
#pragma unroll
    for (int k = 0; k < SPT; ++k) { pos_re[tid * SPT + k] = zr[k]; pos_im[tid * SPT + k] = zi[k]; }
    __syncthreads();
    // fused tail (small grid x N_bins): ring slot of this launch; else slot 0, read by post_gen_kernel, whose previous
    // reader must have finished
    if (!P.tail.st) pdl_wait();
    double2* partial = P.tail.st ? gen_partial_of(P.tail, s_gen) : P.tail.partial + (size_t)blockIdx.x * P.n_bins;
    // positions -> bins: tpb threads per bin (a power of two, consecutive lanes; with few bins a single thread per bin would add
    // span / N_bins values one after the other -- 1 us for 16 bins), each adds every tpb-th position of its bin, then a shuffle tree:
    // a fixed order
    uint32_t tpb = 1;
    while (tpb < 32u && 2u * tpb * P.n_bins <= (uint32_t)kThreads) tpb *= 2u;
    const uint32_t bins_per_pass = (uint32_t)kThreads / tpb;
    for (uint32_t sb0 = 0; sb0 < P.n_bins; sb0 += bins_per_pass) {          // uniform trip count (shuffles below)
        const uint32_t sb = sb0 + (uint32_t)tid / tpb, j = (uint32_t)tid % tpb;
        double re = 0.0, im = 0.0;
        if (sb < P.n_bins)
            for (uint32_t pos = sb + j * P.n_bins; pos < P.span; pos += tpb * P.n_bins) { re += pos_re[pos]; im += pos_im[pos]; }
        for (uint32_t sh = tpb >> 1; sh > 0; sh >>= 1) {
            re += __shfl_xor_sync(0xFFFFFFFFu, re, sh);
            im += __shfl_xor_sync(0xFFFFFFFFu, im, sh);
        }
        if (sb < P.n_bins && j == 0) partial[sb] = make_double2(re, im);
    }
    if (P.tail.st) gen_tail(P.tail, s_gen, reinterpret_cast<double2*>(gen_smem));
}

}  // namespace pcal
