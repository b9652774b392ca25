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
// Mapping: a CTA iteration covers kThreads*SPT consecutive samples (thread t owns samples
// t*SPT .. t*SPT+SPT-1 of it); 65536/(kThreads*SPT) iterations form a tile; tiles are dealt
// round-robin to CTAs.  N_bins must divide kThreads*SPT so every thread keeps fixed bins.
// Per-sample work: decode (2 integer ops) + one packed FFMA2 issue (re and im of two samples).
// fp32 partial sums live for one tile (<= 64 additions), then are added to fp64 accumulators in
// shared memory.
#pragma once
#include "pcal_common.cuh"

namespace pcal {

constexpr uint32_t kTileSamples = 1u << 16;

struct GenParams {
    const void* data;        // [device] packed samples
    uint64_t n_loads;        // complete per-thread loads available (vectors of SPT samples)
    uint64_t n_tiles;
    uint64_t Fs, k0, E, D;   // micro-hertz sample rate; (n0*Foff)%Fs; (tile*Foff)%Fs; (grid*E)%Fs
    uint64_t Foff;
    double2 rho;             // exp(-j w * kThreads*SPT): oscillator step per CTA iteration
    double2 tw[16];          // exp(-j w k), k = 0..15: post-twiddle within a load
    double2* partial;        // [device] [cta][n_bins]
    uint32_t n_bins;
    int sign_mag;
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
template <>
__device__ __forceinline__ void gen_decode<KIND_2BIT>(const uint32_t& v, float* x, int sign_mag) {
    const uint32_t w = sign_mag ? signmag_to_offset_binary(v) : v;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const uint32_t sh = (2 * k <= 21) ? (w << (21 - 2 * k)) : (w >> (2 * k - 21));
        x[k] = __uint_as_float((sh & 0x00600000u) | 0x3F800000u);  // 1 + c/4
    }
}

template <int KIND>
__device__ __forceinline__ typename GenTraits<KIND>::Vec gen_load(const void* base, uint64_t i);
template <> __device__ __forceinline__ uint4 gen_load<KIND_F32>(const void* b, uint64_t i) { return ldg_stream(reinterpret_cast<const uint4*>(b) + i); }
template <> __device__ __forceinline__ uint4 gen_load<KIND_I8>(const void* b, uint64_t i) { return ldg_stream(reinterpret_cast<const uint4*>(b) + i); }
template <> __device__ __forceinline__ uint32_t gen_load<KIND_2BIT>(const void* b, uint64_t i) {
    uint32_t r;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r) : "l"(reinterpret_cast<const uint32_t*>(b) + i));
    return r;
}

template <int KIND>
__global__ void __launch_bounds__(kThreads, 2) gen_kernel(GenParams P) {
    constexpr int SPT = GenTraits<KIND>::SPT;
    constexpr uint32_t SPAN = kThreads * SPT;               // samples per CTA iteration
    constexpr uint32_t ITERS = kTileSamples / SPAN;         // iterations per tile
    constexpr int U = 4;                                     // loads in flight per thread
    using Vec = typename GenTraits<KIND>::Vec;
    extern __shared__ double sacc[];                         // [2*SPT][kThreads] re then im
    const int tid = threadIdx.x;
#pragma unroll
    for (int k = 0; k < 2 * SPT; ++k) sacc[k * kThreads + tid] = 0.0;

    const uint64_t koff = mulmod_u64(P.Foff, (uint64_t)tid * SPT, P.Fs);
    uint64_t k_cta = P.k0 + mulmod_u64(P.E, blockIdx.x, P.Fs);
    if (k_cta >= P.Fs) k_cta -= P.Fs;
    double sphr = 0.0, sphi = 0.0;                           // sum of phasors of valid loads (2-bit)

    for (uint64_t tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
        // ---- resync: exact integer phase -> fp64 phasor ----
        uint64_t k = k_cta + koff;
        if (k >= P.Fs) k -= P.Fs;
        double2 ph = phasor_neg(k, P.Fs);
        k_cta += P.D;
        if (k_cta >= P.Fs) k_cta -= P.Fs;

        float2 ar[SPT / 2], ai[SPT / 2];
#pragma unroll
        for (int k2 = 0; k2 < SPT / 2; ++k2) { ar[k2] = make_float2(0.f, 0.f); ai[k2] = make_float2(0.f, 0.f); }
        float pr = 0.f, pi = 0.f;
        uint64_t li = (tile * ITERS) * kThreads + tid;       // this thread's load index
#pragma unroll 1
        for (uint32_t it = 0; it < ITERS; it += U) {
            Vec v[U];
            bool ok[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                ok[u] = (li + (uint64_t)u * kThreads) < P.n_loads;
                if (ok[u]) v[u] = gen_load<KIND>(P.data, li + (uint64_t)u * kThreads);
            }
            li += (uint64_t)U * kThreads;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const float c = (float)ph.x, s = (float)ph.y;
                if (ok[u]) {
                    float x[SPT];
                    gen_decode<KIND>(v[u], x, P.sign_mag);
                    const float2 cc = make_float2(c, c), ss = make_float2(s, s);
#pragma unroll
                    for (int k2 = 0; k2 < SPT / 2; ++k2) {
                        const float2 xx = make_float2(x[2 * k2], x[2 * k2 + 1]);
                        ffma2(ar[k2], xx, cc);
                        ffma2(ai[k2], xx, ss);
                    }
                    if (KIND == KIND_2BIT) { pr += c; pi += s; }
                }
                // coupled-form oscillator step (eq. 2.6): ph *= rho, fp64
                const double nx = ph.x * P.rho.x - ph.y * P.rho.y;
                const double ny = ph.x * P.rho.y + ph.y * P.rho.x;
                ph.x = nx; ph.y = ny;
            }
        }
        // ---- flush the tile's fp32 sums into the fp64 accumulators ----
#pragma unroll
        for (int k2 = 0; k2 < SPT / 2; ++k2) {
            sacc[(2 * k2) * kThreads + tid] += (double)ar[k2].x;
            sacc[(2 * k2 + 1) * kThreads + tid] += (double)ar[k2].y;
            sacc[(SPT + 2 * k2) * kThreads + tid] += (double)ai[k2].x;
            sacc[(SPT + 2 * k2 + 1) * kThreads + tid] += (double)ai[k2].y;
        }
        sphr += (double)pr; sphi += (double)pi;
    }

    // ---- post-twiddle by exp(-j w k), undo the 2-bit affine code, reduce positions to bins ----
    double zr[SPT], zi[SPT];
#pragma unroll
    for (int k = 0; k < SPT; ++k) {
        double re = sacc[k * kThreads + tid], im = sacc[(SPT + k) * kThreads + tid];
        if (KIND == KIND_2BIT) { re = 8.0 * re - 11.0 * sphr; im = 8.0 * im - 11.0 * sphi; }
        zr[k] = re * P.tw[k].x - im * P.tw[k].y;
        zi[k] = re * P.tw[k].y + im * P.tw[k].x;
    }
    __syncthreads();
    double* pos_re = sacc;                 // [SPAN]
    double* pos_im = sacc + SPAN;          // [SPAN]
#pragma unroll
    for (int k = 0; k < SPT; ++k) { pos_re[tid * SPT + k] = zr[k]; pos_im[tid * SPT + k] = zi[k]; }
    __syncthreads();
    for (uint32_t s = tid; s < P.n_bins; s += kThreads) {
        double re = 0.0, im = 0.0;
        for (uint32_t pos = s; pos < SPAN; pos += P.n_bins) { re += pos_re[pos]; im += pos_im[pos]; }
        P.partial[(size_t)blockIdx.x * P.n_bins + s] = make_double2(re, im);
    }
}

struct GenReduceParams {
    const double2* partial;  // [grid][n_bins]
    double2* P;              // [n_bins] accumulated into
    const uint8_t* tail;     // first byte after the last complete load
    uint64_t n0, n_done, n_total, Fs, Foff;
    uint32_t grid, n_bins;
    int kind, sign_mag;
};

// one thread per bin: fixed-order sum over CTAs, then the ragged tail with exact phases
__global__ void gen_reduce_kernel(GenReduceParams G) {
    const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= G.n_bins) return;
    const uint32_t s = (uint32_t)(((uint64_t)b + G.n_bins - G.n0 % G.n_bins) % G.n_bins);
    double re = 0.0, im = 0.0;
    for (uint32_t c = 0; c < G.grid; ++c) {
        const double2 v = G.partial[(size_t)c * G.n_bins + s];
        re += v.x; im += v.y;
    }
    for (uint64_t t = G.n_done; t < G.n_total; ++t) {
        if ((G.n0 + t) % G.n_bins != b) continue;
        const uint32_t r = (uint32_t)(t - G.n_done);
        double v;
        if (G.kind == KIND_F32) v = (double)reinterpret_cast<const float*>(G.tail)[r];
        else if (G.kind == KIND_I8) v = (double)reinterpret_cast<const int8_t*>(G.tail)[r];
        else {
            const uint32_t code = (G.tail[r >> 2] >> (2 * (r & 3u))) & 3u;
            v = G.sign_mag ? ((code & 2u) ? -(double)(1 + 2 * (code & 1u)) : (double)(1 + 2 * (code & 1u)))
                           : (double)(2 * (int)code - 3);
        }
        const double2 ph = phasor_neg(mulmod_u64(G.Foff, G.n0 + t, G.Fs), G.Fs);
        re += v * ph.x; im += v * ph.y;
    }
    double2 cur = G.P[b];
    cur.x += re; cur.y += im;
    G.P[b] = cur;
}

}  // namespace pcal
