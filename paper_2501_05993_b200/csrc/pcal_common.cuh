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

// Exact division of small numbers by a run-time divisor without the ~150-cycle dependent sequence of a hardware-assisted
// udiv -- the serial tails of the kernels (one CTA, two warps per scheduler) are chains of such latencies.
// q = (x * ceil(2^40 / d)) >> 40 is exact for x * d < 2^40 (here: x < 2^24, d <= 2^12 .. 2^16).  The constant comes from ONE
// fp64 division: 2^40 / d is an integer (d a power of two) or at least 2^-16 away from one, which fp64 resolves (53 bits).
struct FastDiv {
    uint64_t m;
    uint32_t d;
    __device__ __forceinline__ explicit FastDiv(uint32_t div) : m((uint64_t)ceil(1099511627776.0 / (double)div)), d(div) {}
    __device__ __forceinline__ uint32_t div(uint32_t x) const { return (uint32_t)(((uint64_t)x * m) >> 40); }
    __device__ __forceinline__ uint32_t mod(uint32_t x) const { return x - div(x) * d; }
    __device__ __forceinline__ void divmod(uint32_t x, uint32_t& q, uint32_t& r) const { q = div(x); r = x - q * d; }
};

// exp(-j 2 pi k / m) in fp64 for an exactly reduced numerator 0 <= k < m.
__device__ __forceinline__ double2 phasor_neg(uint64_t k, uint64_t m) {
    double s, c;
    sincospi(2.0 * ((double)k / (double)m), &s, &c);
    return make_double2(c, -s);
}

}  // namespace pcal
