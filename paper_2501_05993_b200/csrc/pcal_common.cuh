// pcal_common.cuh -- shared device helpers and geometry constants for libpcal (sm_100a).
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pcal {

// One CTA = 8 warps.  A "vector" is one 16-byte (128-bit) global load; a warp load covers 32
// consecutive vectors = 512 contiguous bytes (4 full 128-byte lines).
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kMaxChannels = 16;      // == PCAL_MAX_CHANNELS of include/pcal.h
constexpr int kUnroll = 8;            // independent 128-bit loads in flight per thread

// sample kinds handled by the kernels
enum Kind : int { KIND_F32 = 0, KIND_I8 = 1, KIND_2BIT = 2 };

// Streaming 128-bit load: read-only path, do not allocate in L1 (each byte is used once).
__device__ __forceinline__ uint4 ldg_stream(const uint4* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

// Programmatic dependent launch (see launch_chain in pcal_api.cu).  pdl_release(): first statement of
// every kernel of the per-step chain -- the successor's CTAs may be scheduled behind this grid.
// pdl_wait(): returns once the predecessor grid has COMPLETED and its writes are visible; a kernel
// calls it before its first access to memory that any earlier kernel of the chain reads or writes.
// Since a grid cannot complete before its own pdl_wait() has returned, completion is transitive along
// the chain no matter how early the release is issued.  The streaming kernels (fold_*, gen_kernel)
// only read the caller's input before the wait, so their load phase overlaps the small kernels of the
// previous step/segment.  Both are no-ops when the kernel was launched in plain stream order.
__device__ __forceinline__ void pdl_release() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ uint32_t lop3_xor3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t lop3_maj(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}

// Carry-save adder on 32 independent bit columns: a + b + c = s + 2*cy (per bit).
// For words made of 2-bit fields (value = lo + 2*hi) the identity carries over to field values:
// val(a)+val(b)+val(c) = val(s) + 2*val(cy)  -- two LOP3 compress three packed words into two.
__device__ __forceinline__ void csa(uint32_t a, uint32_t b, uint32_t c, uint32_t& s, uint32_t& cy) {
    s = lop3_xor3(a, b, c);
    cy = lop3_maj(a, b, c);
}

// SIGN_MAG code (s<<1)|m  ->  OFFSET_BINARY code c' with level = 2c'-3:
//   c' = x ^ 0b10 ^ (s ? 0b01 : 0)   for every 2-bit field at once (one shift + one LOP3).
__device__ __forceinline__ uint32_t signmag_to_offset_binary(uint32_t x) {
    return x ^ 0xAAAAAAAAu ^ ((x >> 1) & 0x55555555u);
}

__device__ __forceinline__ uint32_t word_of(const uint4& v, int j) {
    return j == 0 ? v.x : (j == 1 ? v.y : (j == 2 ? v.z : v.w));
}

// (a * b) mod m for a, b < m < 2^63 without 128-bit division: double-and-add (64 steps worst case).
// Only used a handful of times per kernel (tails, per-CTA start phases).
__device__ __forceinline__ uint64_t mulmod_u64(uint64_t a, uint64_t b, uint64_t m) {
    uint64_t r = 0;
    if (a >= m) a %= m;                                     // callers usually pass an already reduced factor
    if (__umul64hi(a, b) == 0) return (a * b) % m;       // the product fits in 64 bits (the usual case: small multipliers)
    while (b) {
        if (b & 1) { r += a; if (r >= m) r -= m; }
        a += a; if (a >= m) a -= m;
        b >>= 1;
    }
    return r;
}

// exp(-j 2 pi k / m) in fp64 for an exactly reduced numerator 0 <= k < m.
__device__ __forceinline__ double2 phasor_neg(uint64_t k, uint64_t m) {
    double s, c;
    sincospi(2.0 * ((double)k / (double)m), &s, &c);
    return make_double2(c, -s);
}

}  // namespace pcal

// ---- calibration: a pure streaming read of `n_vec` 16-byte vectors (no decode, no fold) --------
// Same load instruction, block size and software pipelining as the fold kernels; what it reaches
// on a given buffer size is the practical ceiling for any read-once kernel of that size
// (bench.py reports it beside the roofline fraction).  The xor of all words lands in out[0] only
// if it equals a magic value, so the loads cannot be optimised away.
namespace pcal {
__global__ void __launch_bounds__(kThreads, 3) read_probe_kernel(const uint4* __restrict__ d, uint64_t n_vec, uint32_t* out) {
    pdl_release();
    const uint64_t stride = (uint64_t)gridDim.x * kThreads;
    uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    uint32_t acc = 0;
    uint4 v[4], w[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const uint64_t a = i + u * stride; v[u] = a < n_vec ? ldg_stream(d + a) : make_uint4(0, 0, 0, 0); }
    for (i += 4 * stride; i < n_vec + 4 * stride; i += 4 * stride) {
#pragma unroll
        for (int u = 0; u < 4; ++u) { const uint64_t a = i + u * stride; w[u] = a < n_vec ? ldg_stream(d + a) : make_uint4(0, 0, 0, 0); }
#pragma unroll
        for (int u = 0; u < 4; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = w[u];
    }
    if (acc == 0x5ca1ab1eu) out[0] = acc;
}

// ---- calibration: issue-rate ceilings of the pipes the kernels lean on ----------------
// kind 0: FFMA (fp32 FMA pipe), 1: LOP3 (integer/logic pipe), 2: IMMA m16n8k16 s8 (legacy tensor path used by
// gen_mma_kernel).  Eight independent dependency chains per thread, `iters` trips; the result is written so that
// nothing is optimised away.  The host times the launch and reports instructions per second.
template <int KIND_P>
__global__ void __launch_bounds__(kThreads) pipe_probe_kernel(uint32_t iters, uint32_t* out) {
    uint32_t a[8];
    float f[8];
    int d[8][4];
#pragma unroll
    for (int j = 0; j < 8; ++j) { a[j] = threadIdx.x * 2654435761u + j; f[j] = 1.0f + j; d[j][0] = d[j][1] = d[j][2] = d[j][3] = 0; }
    const float m = 1.0000001f, q = 1e-9f;
    const uint32_t x = blockIdx.x | 0x01010101u, y = threadIdx.x * 0x01010101u;
    for (uint32_t i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (KIND_P == 0) f[j] = __fmaf_rn(f[j], m, q);
            else if (KIND_P == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[j]) : "r"(x), "r"(y));
            else asm volatile("mma.sync.aligned.m16n8k16.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
                              : "+r"(d[j][0]), "+r"(d[j][1]), "+r"(d[j][2]), "+r"(d[j][3]) : "r"(x), "r"(y), "r"(a[j]));
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j] + __float_as_uint(f[j]) + (uint32_t)(d[j][0] + d[j][1] + d[j][2] + d[j][3]);
    if (s == 0x5ca1ab1eu) out[0] = s;
}

}  // namespace pcal
