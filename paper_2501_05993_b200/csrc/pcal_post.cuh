// pcal_post.cuh -- the small deterministic kernels behind the hot loop:
//   reduce_replicas_kernel  per-CTA partials of the fold kernels -> one sum per (slot, field, lane)
//                       (the "binary tree stepping" the paper leaves to the host)
//   rotate_fold_kernel  A[r] * exp(-j w_off r) folded to N_bins (eq. 2.3 + 2.2 after the reordering
//                       of PAPER.md:200), ragged tail (< 1 vector), accumulate into the context
//   post_gen_kernel     per-CTA generator partials -> bins, ragged tail, accumulate (large N_bins; else pcal_gen_tail.cuh)
//   dft_kernel          T[i] = sum_b P[b] exp(-j 2 pi i b / N_bins)
// All sums run in a fixed order (no floating-point atomics): two runs give bit-identical results.
#pragma once
#include "pcal_common.cuh"

namespace pcal {

constexpr int kPostThreads = 256;

// Progress counters of a context whose fold kernels run the fused tail (pcal_tail.cuh, "Pipelining").
struct TailState {
    unsigned long long tick;  // tickets taken (one per CTA of every fold launch)
    uint32_t n_done;          // fold launches whose stage C has finished
    uint32_t dft_started;     // CTAs of DFT kernels that have started ...
    uint32_t dft_finished;    // ... and that have finished reading P
    uint32_t pad;
};


// ---- stage 1: sum the R replicas of every slot group -------------------------------------------
// in : elem partial[(rho*q + p)][F][32]          out: double val[p][F][32]
// For 2-bit data the partials are code sums; val = 2*sum - 3*(vectors folded into this slot) is the
// level sum.  Integer sums are exact in a double (|val| < 2^53).  One thread per element; the
// replica loads are issued eight at a time and added in replica order (deterministic for fp64).
struct ReplicaParams {
    const void* partial;
    double* val;
    uint32_t q, R, F, ns;        // ns: replica slices per element (1, 2, 4 or 8)
    uint32_t cnt_quot, cnt_rem;   // vectors per slot: cnt_quot + (p*32 + lane < cnt_rem)
    int kind;
};

// replicas r = first, first + step, ... < R, eight loads in flight, added in replica order
template <typename Tin, typename Tacc>
__device__ __forceinline__ Tacc replica_sum(const Tin* src, size_t stride, uint32_t first, uint32_t step, uint32_t R) {
    Tacc a = 0;
    for (uint32_t r0 = first; r0 < R; r0 += 8 * step) {
        Tin t[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) t[k] = (r0 + k * step < R) ? __ldcg(src + (size_t)(r0 + k * step) * stride) : (Tin)0;
#pragma unroll
        for (int k = 0; k < 8; ++k) a += (Tacc)t[k];
    }
    return a;
}

// A CTA serves 256/ns consecutive elements with ns replica slices (ns = 1, 2, 4 or 8, chosen by
// the host so that a slice has at most ~8 replicas): thread = (slice, element), consecutive
// threads read consecutive elements (coalesced); the slice sums are then added in slice order.
__global__ void __launch_bounds__(kPostThreads) reduce_replicas_kernel(ReplicaParams P) {
    pdl_release();
    pdl_wait();
    __shared__ double sd[kPostThreads];
    __shared__ long long si[kPostThreads];
    const uint32_t E = P.F * 32u, total = P.q * E;          // a multiple of 128 (float32, odd q: not of 256)
    const uint32_t epc = kPostThreads / P.ns;                // elements per CTA
    const uint32_t sl = threadIdx.x / epc, e = threadIdx.x % epc;
    const uint32_t i = blockIdx.x * epc + e;
    const bool in = i < total;                               // (the last CTA may be partly empty)
    if (!in) { sd[threadIdx.x] = 0.0; si[threadIdx.x] = 0; }
    else if (P.kind == KIND_F32) sd[threadIdx.x] = replica_sum<double, double>(reinterpret_cast<const double*>(P.partial) + i, total, sl, P.ns, P.R);
    else if (P.kind == KIND_I8) si[threadIdx.x] = replica_sum<int32_t, long long>(reinterpret_cast<const int32_t*>(P.partial) + i, total, sl, P.ns, P.R);
    else si[threadIdx.x] = replica_sum<uint16_t, long long>(reinterpret_cast<const uint16_t*>(P.partial) + i, total, sl, P.ns, P.R);
    __syncthreads();
    if (sl != 0 || !in) return;
    double v;
    if (P.kind == KIND_F32) {
        v = 0.0;
        for (uint32_t k = 0; k < P.ns; ++k) v += sd[k * epc + e];
    } else {
        long long a = 0;
        for (uint32_t k = 0; k < P.ns; ++k) a += si[k * epc + e];
        if (P.kind == KIND_2BIT) {
            const uint32_t vslot = (i / E) * 32u + (i & 31u);
            a = 2 * a - 3ll * (long long)(P.cnt_quot + (vslot < P.cnt_rem ? 1u : 0u));
        }
        v = (double)a;
    }
    P.val[i] = v;
}

// ---- stage 2: rotate and fold to N_bins --------------------------------------------------------
struct RotateParams {
    const double* val;        // [device] val[q][F][32] from stage 1
    const double2* lut;       // [device] concatenated per-channel rotator tables (eq. 2.4)
    const uint32_t* lut_off;  // [device] per channel: first entry
    const uint32_t* lut_len;  // [device] per channel: N_rotator,c (1 => no rotation)
    double2* P;               // [device] folded bins [C][N_bins]
    long long* Pint;          // [device] exact integer bins [C][N_bins]
    const uint8_t* tail;      // [device] first byte after the last complete vector
    uint64_t n0;              // absolute index of the first sample of this piece
    uint64_t NT;              // time samples covered by complete vectors
    uint64_t n_total;         // time samples in this piece
    uint32_t q, F, C;         // slot groups, fields per vector, channels
    uint32_t spv, spv_log2;   // time samples per vector (power of two)
    uint32_t n_bins;
    uint32_t tpp;             // threads per (channel, bin) pair: 32 (a warp) or 256 (the CTA)
    uint32_t have_val;        // 0 when the piece has no complete vector
    int kind;                 // KIND_*
    int sign_mag;
    int integer_exact;        // every channel unrotated and integer input: keep Pint
    int overwrite;            // first piece after reset: P = new instead of P += new
    int release_late;         // do not let the dependent grid start early (its stage C reads P without a grid-wide wait)
};

__device__ __forceinline__ double decode_tail(int kind, int sign_mag, const uint8_t* tail, uint32_t t, uint32_t c, uint32_t C) {
    if (kind == KIND_F32) return (double)reinterpret_cast<const float*>(tail)[t];
    if (kind == KIND_I8) return (double)reinterpret_cast<const int8_t*>(tail)[t];
    const uint32_t bit = (t * C + c) * 2u;
    const uint32_t code = (tail[bit >> 3] >> (bit & 7u)) & 3u;
    if (sign_mag) return (code & 2u) ? -(double)(1 + 2 * (code & 1u)) : (double)(1 + 2 * (code & 1u));
    return (double)(2 * (int)code - 3);
}

// The super-row (q*32 vectors = SR time samples, a multiple of the fold period and of N_bins) is
// the index space of val: offset o in [0, SR) <-> slot group o / (32 spv), lane, time-in-vector.
// Bin b of channel c collects the offsets o = o_b + j*N_bins.  A pair is served by `tpp` threads:
// thread u adds its elements j = u, u + tpp, ... in order (four look-ups in flight), then the
// lane sums are combined by a fixed butterfly (and, for tpp = 256, the 8 warp sums in warp order).
__global__ void __launch_bounds__(kPostThreads) rotate_fold_kernel(RotateParams P) {
    if (!P.release_late) pdl_release();
    pdl_wait();
    __shared__ double sre[kPostThreads / 32], sim[kPostThreads / 32];
    __shared__ long long sint[kPostThreads / 32];
    const uint32_t tid = threadIdx.x, lane = tid & 31u, w = tid >> 5;
    const uint32_t pairs = P.C * P.n_bins;
    const uint32_t ppc = kPostThreads / P.tpp;                  // pairs per CTA: 8 or 1
    const uint32_t pp = blockIdx.x * ppc + (P.tpp == 32 ? w : 0);
    const bool active = pp < pairs;                              // uniform per warp
    const uint32_t u = P.tpp == 32 ? lane : tid;
    const uint32_t c = active ? pp / P.n_bins : 0, b = active ? pp % P.n_bins : 0;
    const uint32_t L = P.lut_len[c];
    const double2* lut = P.lut + P.lut_off[c];
    const uint32_t SR = P.q * 32u * P.spv;
    double are = 0.0, aim = 0.0;
    long long ai = 0;
    if (active && P.have_val) {
        const uint32_t E = P.F * 32u, span_log2 = 5u + P.spv_log2;
        const uint32_t o_b = (uint32_t)(((uint64_t)b + P.n_bins - (P.n0 % P.n_bins)) % P.n_bins);
        uint32_t o = o_b + u * P.n_bins;
        const uint32_t ostep = P.tpp * P.n_bins;
        auto at = [&](uint32_t oo) -> uint32_t {   // element index of super-row offset oo, channel c
            const uint32_t p = oo >> span_log2, d = oo & ((1u << span_log2) - 1u);
            return p * E + (((d & (P.spv - 1u)) * P.C + c) << 5) + (d >> P.spv_log2);
        };
        if (L > 1) {
            uint32_t k = (uint32_t)((P.n0 % L + o) % L);
            const uint32_t kstep = ostep % L;
            for (; o < SR; o += 4u * ostep) {
                double2 ph[4];
                double v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t oo = o + j * ostep;
                    const bool ok = oo < SR;
                    ph[j] = ok ? __ldg(lut + k) : make_double2(0.0, 0.0);
                    v[j] = ok ? __ldcg(P.val + at(oo)) : 0.0;
                    k += kstep; if (k >= L) k -= L;
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) { are += v[j] * ph[j].x; aim += v[j] * ph[j].y; }
            }
        } else {
            for (; o < SR; o += 4u * ostep) {
                double v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) { const uint32_t oo = o + j * ostep; v[j] = (oo < SR) ? __ldcg(P.val + at(oo)) : 0.0; }
#pragma unroll
                for (int j = 0; j < 4; ++j) { are += v[j]; ai += (long long)v[j]; }
            }
        }
    }
#pragma unroll
    for (uint32_t s = 16; s > 0; s >>= 1) {
        are += __shfl_xor_sync(0xFFFFFFFFu, are, s);
        aim += __shfl_xor_sync(0xFFFFFFFFu, aim, s);
        ai += __shfl_xor_sync(0xFFFFFFFFu, ai, s);
    }
    if (P.tpp != 32) {
        if (lane == 0) { sre[w] = are; sim[w] = aim; sint[w] = ai; }
        __syncthreads();
        are = 0.0; aim = 0.0; ai = 0;
#pragma unroll
        for (int ww = 0; ww < kPostThreads / 32; ++ww) { are += sre[ww]; aim += sim[ww]; ai += sint[ww]; }
        if (tid != 0) return;
    } else if (lane != 0) {
        return;
    }
    if (!active) return;
    const uint32_t n_tail = (uint32_t)(P.n_total - P.NT);
    if (n_tail) {   // ragged tail: samples NT .. n_total-1 (fewer than one vector)
        uint32_t bb = (uint32_t)((P.n0 + P.NT) % P.n_bins);
        uint32_t k = L > 1 ? (uint32_t)((P.n0 + P.NT) % L) : 0;
        for (uint32_t t = 0; t < n_tail; ++t) {
            if (bb == b) {
                const double v = decode_tail(P.kind, P.sign_mag, P.tail, t, c, P.C);
                if (L > 1) { const double2 ph = lut[k]; are += v * ph.x; aim += v * ph.y; }
                else { are += v; ai += (long long)v; }
            }
            if (++bb == P.n_bins) bb = 0;
            if (L > 1 && ++k == L) k = 0;
        }
    }
    if (!P.overwrite) {
        const double2 cur = P.P[pp];
        are += cur.x; aim += cur.y;
        if (P.integer_exact) ai += P.Pint[pp];
    }
    P.P[pp] = make_double2(are, aim);
    if (P.integer_exact) P.Pint[pp] = ai;
}

// ---- generator path, un-fused (large grid x N_bins: pcal_gen_tail.cuh explains): per-CTA partial bins -> context bins ------------------------------------
struct GenPostParams {
    const double2* partial;  // [device] [grid][n_bins], bin index relative to the piece start
    double2* P;              // [device] [n_bins] accumulated into (or overwritten)
    const uint8_t* tail;     // [device] first byte after the last complete load
    uint64_t n0, n_done, n_total, Fs, Foff;
    uint32_t grid, n_bins;
    int kind, sign_mag, overwrite;
};

// One CTA per 32 consecutive bins: warp w sums the CTAs w, w+8, ... (coalesced 512-byte rows),
// the 8 warp sums are added in warp order, then the ragged tail with exactly reduced phases.
__global__ void __launch_bounds__(kPostThreads) post_gen_kernel(GenPostParams G) {
    pdl_release();
    pdl_wait();
    __shared__ double sre[kPostThreads / 32][32], sim[kPostThreads / 32][32];
    const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const uint32_t b = blockIdx.x * 32u + lane;
    const bool ok = b < G.n_bins;
    const uint32_t shift = (uint32_t)(G.n0 % G.n_bins);
    const uint32_t s = ok ? (b + G.n_bins - shift) % G.n_bins : 0;
    double re = 0.0, im = 0.0;
    if (ok) {
        constexpr uint32_t W = kPostThreads / 32;
        for (uint32_t c0 = w; c0 < G.grid; c0 += 8u * W) {        // eight loads in flight, added in CTA order
            double2 v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = (c0 + k * W < G.grid) ? __ldcg(G.partial + (size_t)(c0 + k * W) * G.n_bins + s) : make_double2(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < 8; ++k) { re += v[k].x; im += v[k].y; }
        }
    }
    sre[w][lane] = re; sim[w][lane] = im;
    __syncthreads();
    if (w != 0 || !ok) return;
    re = 0.0; im = 0.0;
#pragma unroll
    for (int ww = 0; ww < kPostThreads / 32; ++ww) { re += sre[ww][lane]; im += sim[ww][lane]; }
    const uint32_t n_tail = (uint32_t)(G.n_total - G.n_done);
    if (n_tail) {
        const uint32_t bb0 = (uint32_t)((G.n0 + G.n_done) % G.n_bins);        // bin of tail sample 0
        for (uint32_t t = (b + G.n_bins - bb0) % G.n_bins; t < n_tail; t += G.n_bins) {   // this bin's tail samples, in order
            const double v = decode_tail(G.kind, G.sign_mag, G.tail, t, 0, 1);
            const double2 ph = phasor_neg(mulmod_u64(G.Foff, G.n0 + G.n_done + t, G.Fs), G.Fs);
            re += v * ph.x; im += v * ph.y;
        }
    }
    if (!G.overwrite) { const double2 cur = G.P[b]; re += cur.x; im += cur.y; }
    G.P[b] = make_double2(re, im);
}

// ---- DFT of the folded period ------------------------------------------------------------------
// T[c][i] = sum_b P[c][b] * W[(i'*b) mod N], i' = (i - k_shift) mod N, W[k] = exp(-j 2 pi k/N)
// (twiddle table built on the host in long double).  One warp per output (opw outputs in turn, so
// that the grid stays small: its CTAs share the SMs with the streaming kernel of the next step): lane l
// sums the terms b = l, l+32, ... in order, then a fixed xor-butterfly adds the 32 lane sums.  The
// twiddle index is stepped in integers, never formed as a floating-point angle.
constexpr int kDftThreads = 256;
__global__ void __launch_bounds__(kDftThreads) dft_kernel(const double2* __restrict__ P, const double2* __restrict__ W,
                                                          double2* __restrict__ T, double2* __restrict__ T_host,
                                                          uint32_t N, uint32_t k_shift, uint32_t opw, TailState* st, int finish_late) {
    if (st) {   // counted before the dependents may start: a later fold kernel waits for these CTAs to have read P
        if (threadIdx.x == 0) atomicAdd(&st->dft_started, 1u);
        __syncthreads();
    }
    pdl_release();
    pdl_wait();
    extern __shared__ double2 dft_sm[];  // [N] bins of this channel, [N] twiddles
    double2* sp = dft_sm;
    double2* sw = dft_sm + N;
    const uint32_t c = blockIdx.y;
    for (uint32_t t = threadIdx.x; t < N; t += kDftThreads) {
        sp[t] = __ldcg(P + (size_t)c * N + t);      // L2: the producer grid may have overlapped this one
        sw[t] = W[t];
    }
    __syncthreads();
    // P has been read.  (finish_late: contexts whose fold kernel may itself deliver T count this CTA out only after
    // its T writes, so that a later launch cannot be overtaken by them.)
    if (st && !finish_late && threadIdx.x == 0) { __threadfence(); atomicAdd(&st->dft_finished, 1u); }
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t i0 = (blockIdx.x * (kDftThreads / 32) + (threadIdx.x >> 5)) * opw;
    for (uint32_t i = i0; i < i0 + opw && i < N; ++i) {       // whole warp together
        const uint32_t ii = (i + N - k_shift % N) % N;
        uint32_t k = (uint32_t)(((uint64_t)ii * lane) % N);
        const uint32_t kstep = (uint32_t)(((uint64_t)ii * 32u) % N);
        double re = 0.0, im = 0.0;
        for (uint32_t b = lane; b < N; b += 32u) {
            const double2 p = sp[b], w = sw[k];
            re += p.x * w.x - p.y * w.y;
            im += p.x * w.y + p.y * w.x;
            k += kstep; if (k >= N) k -= N;
        }
#pragma unroll
        for (uint32_t s = 16; s > 0; s >>= 1) {
            re += __shfl_xor_sync(0xFFFFFFFFu, re, s);
            im += __shfl_xor_sync(0xFFFFFFFFu, im, s);
        }
        if (lane == 0) {
            T[(size_t)c * N + i] = make_double2(re, im);
            if (T_host) T_host[(size_t)c * N + i] = make_double2(re, im);   // mapped pinned host memory
        }
    }
    if (st && finish_late) {
        __syncthreads();
        if (threadIdx.x == 0) { __threadfence(); atomicAdd(&st->dft_finished, 1u); }
    }
}

// ---- the same DFT inside a CTA that already holds P in shared memory (fused tails) ----------------------------
// T[c][i] = X_c[(i - k_shift) mod N], X_c[k] = sum_b P[c][b] W[(k b) mod N], evaluated in two stages for N = N1 N2 (N1 = 1:
// the plain sum): with b = N2 b1 + b2 and k = k1 + N1 k2,
//     Y[k1][b2] = W[(k1 b2) mod N] * sum_{b1 < N1} P[N2 b1 + b2] W[(N2 k1 b1) mod N]
//     X[k1 + N1 k2] = sum_{b2 < N2} Y[k1][b2] W[(N1 k2 b2) mod N]
// -- N (N1 + N2) complex MACs per channel instead of N^2, every twiddle taken from the table at an index reduced in
// integers, every sum in a fixed order.  All n_ch channels at once (one thread per output).  sP, sY: [n_ch][N] each in
// shared memory (sY is scratch, laid out [b2][k1] per channel); all threads of the CTA call it.  With sOut != null the tones
// are left there ([n_ch][N] in shared memory; may be sP) instead of being stored, for a caller that is not yet allowed to.
__device__ __forceinline__ void dft_in_cta(const double2* sP, double2* sY, const double2* __restrict__ W, uint32_t n_ch, uint32_t N,
                                           uint32_t N1, uint32_t k_shift, double2* T_dev, double2* T_host, uint32_t nthreads,
                                           double2* sOut = nullptr) {
    const uint32_t N2 = N / N1, tid = threadIdx.x, total = n_ch * N;
    const FastDiv dN(N), dN1(N1), dN2(N2);                 // (indices below 2^24, divisors <= 4096)
    // sum_{j < n} x[j * stride] * W[(j * step) mod N] in index order; eight loads of each operand in flight at a time
    auto dot = [&](const double2* x, uint32_t stride, uint32_t n, uint32_t step, double& re, double& im) {
        uint32_t idx = 0;
        re = 0.0; im = 0.0;
        for (uint32_t j0 = 0; j0 < n; j0 += 8u) {
            double2 xv[8], wv[8];
#pragma unroll
            for (uint32_t j = 0; j < 8u; ++j) {
                const bool in = j0 + j < n;
                xv[j] = in ? x[(j0 + j) * stride] : make_double2(0.0, 0.0);
                wv[j] = in ? __ldg(W + idx) : make_double2(0.0, 0.0);
                idx += step; if (idx >= N) idx -= N;
            }
#pragma unroll
            for (uint32_t j = 0; j < 8u; ++j) {
                re += xv[j].x * wv[j].x - xv[j].y * wv[j].y;
                im += xv[j].x * wv[j].y + xv[j].y * wv[j].x;
            }
        }
    };
    for (uint32_t oo = tid; oo < total; oo += nthreads) {
        uint32_t c, o, k1, b2;
        dN.divmod(oo, c, o);
        dN2.divmod(o, k1, b2);
        double re, im;
        dot(sP + c * N + b2, N2, N1, dN.mod(N2 * k1), re, im);
        const double2 w = __ldg(W + dN.mod(k1 * b2));
        sY[c * N + b2 * N1 + k1] = make_double2(re * w.x - im * w.y, re * w.y + im * w.x);
    }
    __syncthreads();
    for (uint32_t oo = tid; oo < total; oo += nthreads) {
        uint32_t c, o, k1, k2;
        dN.divmod(oo, c, o);
        dN1.divmod(o, k2, k1);
        double re, im;
        dot(sY + c * N + k1, N1, N2, dN.mod(N1 * k2), re, im);
        const uint32_t i = c * N + dN.mod(o + k_shift);
        if (sOut) { sOut[i] = make_double2(re, im); continue; }
        T_dev[i] = make_double2(re, im);
        if (T_host) T_host[i] = make_double2(re, im);
    }
    __syncthreads();
}

__global__ void zero_kernel(double2* P, long long* Pint, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { P[i] = make_double2(0.0, 0.0); Pint[i] = 0; }
}

// P[i] = sum_r parts[r][i], r = 0 .. n_parts-1 in that order (the exchange step of a time-sharded run)
// (Pint, when given: the exact integer bins of unrotated integer input -- the real parts are integers below 2^53, so the
//  fp64 sums above are exact and llrint recovers them)
__global__ void sum_parts_kernel(double2* P, long long* Pint, const double2* parts, uint32_t n, uint32_t n_parts) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double re = 0.0, im = 0.0;
    for (uint32_t r = 0; r < n_parts; ++r) { const double2 v = parts[(size_t)r * n + i]; re += v.x; im += v.y; }
    P[i] = make_double2(re, im);
    if (Pint) Pint[i] = llrint(re);
}

__global__ void add_bins_kernel(double2* P, long long* Pint, const double2* add, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { P[i].x += add[i].x; P[i].y += add[i].y; if (Pint) Pint[i] = llrint(P[i].x); }
}

}  // namespace pcal
