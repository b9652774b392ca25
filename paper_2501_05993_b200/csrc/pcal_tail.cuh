// pcal_tail.cuh -- the reduction behind the fold kernels, run INSIDE the fold kernel by the CTAs that
// finish last ("fused tail"): a5 of SURVEY section 8 (deterministic reduction of per-block partials;
// the step the paper leaves to the host CPU) plus the one-off rotation by the
// table of eq. 2.4 after the reordering of PAPER.md:200.
//
// Same arithmetic as reduce_replicas_kernel + rotate_fold_kernel (pcal_post.cuh), which remain as the
// un-fused path for geometries the tail does not take (`fused` in pcal_api.cu's prepare).  Three stages, each
// entered by exactly one CTA per group, elected by an arrival counter (every CTA: write partial, barrier,
// one atom.add.acq_rel by one thread; the CTA that observes count-1 is last and reads what the others
// wrote):
//   A  last CTA of slot group p: sum the R replica partials of the group (replica order), code sums
//      -> level sums, into shared memory                                   [F*32 values]
//   B  same CTA: multiply by the rotator table and fold the group's 32*spv time samples into per-group
//      bins G[p][c][b]   (fixed thread -> element map + fixed butterfly: deterministic)
//   C  last CTA of the grid: P[c][b] (+)= sum_p G[p][c][b] in group order, ragged tail (< 1 vector)
//      added, integer bins kept when the data is integer and unrotated; counters reset for the next
//      launch; for pcal_integrate / pcal_extract_series with N_bins <= 64 also the DFT.
// A step of the LUT path is thereby ONE launch (plus the DFT kernel of pcal_finalize for larger N_bins).
//
// Pipelining across launches.  Partials, counters and G live in a ring of kTailSlots slots and a fold
// kernel never executes griddepcontrol.wait.  Every CTA takes a ticket (64-bit atomicAdd on the
// context's TailState) BEFORE it lets the dependent grid be scheduled; a dependent grid starts only
// after every CTA of its predecessor has done so, hence all tickets of one launch are taken before any
// CTA of a later launch runs and s = ticket / gridDim.x is the launch's sequence number -- derived on the
// device, so launches replayed from a CUDA graph (frozen parameters) stay correct.  Launch s uses slot
// s mod kTailSlots.  Three conditions replace the grid-wide wait, each checked by one thread with an
// acquire load (spinning only if ever needed; the grids waited for were dispatched earlier, so they
// make progress):
//   before the partial writes   n_done >= s - kTailSlots + 1   (the slot's previous user finished stage C)
//   before stage C              n_done == s                    (P holds every earlier launch, in order)
//   before stage C              dft_finished >= X              (every earlier DFT kernel has read P; X =
//                               dft_started as seen before this CTA released its dependents, i.e. the
//                               CTAs of all DFT kernels that precede this launch in the stream)
// and stage C ends by publishing n_done = s + 1.  Consecutive launches therefore overlap completely
// except for stage C, and HBM never drains at a kernel boundary.  Kernels that follow in plain stream
// order (and the DFT kernel, which waits for its predecessor grid) see the finished accumulators.
#pragma once
#include <cstddef>
#include "pcal_post.cuh"

namespace pcal {

struct TailParams {
    uint32_t* cnt;            // [device] [slot][q+2] arrival counters (groups, grid, finishers), zero between launches
    double2* G;               // [device] [slot][q][C*n_bins] per-group bins
    const double2* lut;       // [device] concatenated per-channel rotator tables (eq. 2.4)
    uint32_t lut_off[kMaxChannels];  // per channel: first entry (by value: no dependent load in the serial tail)
    uint32_t lut_len[kMaxChannels];  // per channel: N_rotator,c (1 => no rotation)
    double2* P;               // [device] folded bins [C][N_bins]
    long long* Pint;          // [device] exact integer bins [C][N_bins]
    const uint8_t* tail;      // [device] first byte after the last complete vector
    uint64_t n0, NT, n_total; // absolute index of the first sample; samples in whole vectors; samples in the piece
    uint32_t n0_mod_bins;     // n0 mod N_bins
    uint32_t n0_mod_L[kMaxChannels];   // n0 mod N_rotator,c
    uint32_t cnt_quot, cnt_rem;   // vectors per slot: cnt_quot + (p*32 + lane < cnt_rem)
    uint32_t C, spv, spv_log2, n_bins;
    uint32_t tpp;             // threads per (channel, bin) pair in stage B: power of two <= 32
    int kind, sign_mag, integer_exact, overwrite;
    int enabled;              // 0: the caller launches reduce_replicas_kernel + rotate_fold_kernel instead
    TailState* st;            // [device] tickets and progress counters of the context
    uint64_t partial_stride;  // bytes between the partial buffers of consecutive slots
    // pcal_integrate on small periods: stage C also takes the N_bins-point DFT and delivers T
    int fuse_dft;             // 1: the DFT is cheap in two stages and (C + 1) * N_bins complex values fit in the scratch
    uint32_t dft_n1;          // N_bins = dft_n1 * N2 (dft_in_cta, pcal_post.cuh)
    uint32_t k_shift;
    const double2* W;         // [device] exp(-j 2 pi k / N_bins), k < N_bins
    double2* T_dev;           // [device] tone spectrum [C][N_bins]
    double2* T_host;          // device-visible pinned host memory or null
    double2* P_copy;          // [device] second destination of the folded bins (time series output) or null
};

constexpr uint32_t kTailSlots = 8;
constexpr uint32_t kTailFinishers = 8;      // CTAs that share stage C of the fused tail

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// n_done and dft_started of a context in ONE acquire load (they share an aligned 64-bit word): the ticket thread of every launch
// reads both before it takes its ticket, and each dependent global round trip there is ~0.7 us on the launch's critical path
static_assert(offsetof(TailState, n_done) == 8 && offsetof(TailState, dft_started) == 12, "n_done | dft_started: one 64-bit word");
__device__ __forceinline__ void ld_acquire_done_started(const TailState* st, uint32_t& done, uint32_t& started) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(&st->n_done) : "memory");
    done = (uint32_t)v; started = (uint32_t)(v >> 32);
}
__device__ __forceinline__ void st_release_u32(uint32_t* p, uint32_t v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Arrival on an election counter: release (everything this CTA wrote before the preceding barrier) and
// acquire (what the earlier arrivals released) in one instruction, issued by one thread per CTA.
__device__ __forceinline__ uint32_t arrive_acq_rel(uint32_t* p) {
    uint32_t v;
    asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Called by every thread of a fold kernel once its first loads are in flight: ticket, then the dependent
// grid may be scheduled.  s_gen (shared): [0] = sequence number s of this launch, [1] = X (see above),
// [2] = 1 when the slot was already free at that time (the usual case: nothing to check later).
__device__ __forceinline__ void fold_ticket_and_release(const TailParams& T, uint32_t* s_gen) {
    if (T.enabled) {
        if (threadIdx.x == 0) {
            // (the ticket first, the acquire load behind it: both are in flight together -- one round trip, not two; X only has to
            //  be read before this CTA releases its dependents, see above)
            const unsigned long long tk = atomicAdd(&T.st->tick, 1ull);
            uint32_t done, x;
            ld_acquire_done_started(T.st, done, x);
            const uint32_t seq = (uint32_t)(tk / gridDim.x);
            s_gen[0] = seq; s_gen[1] = x;
            s_gen[2] = ((int32_t)(done - (seq - kTailSlots + 1u)) >= 0) ? 1u : 0u;
        }
        __syncthreads();      // thread 0 holds the ticket (it stored the quotient) before any thread releases
    }
    pdl_release();
}

// Called by every thread of a fold kernel after its loads and before its partial writes.
__device__ __forceinline__ void fold_wait_slot(const TailParams& T, const uint32_t* s_gen) {
    if (T.enabled) {
        if (threadIdx.x == 0 && !s_gen[2])
            while ((int32_t)(ld_acquire_u32(&T.st->n_done) - (s_gen[0] - kTailSlots + 1u)) < 0) __nanosleep(64);
        __syncthreads();
    } else {
        pdl_wait();   // the partials of the previous launch may still be read by its reduce kernel
    }
}

// this launch's partial buffer
__device__ __forceinline__ void* fold_partial_of(const TailParams& T, void* base, const uint32_t* s_gen) {
    return T.enabled ? reinterpret_cast<uint8_t*>(base) + (uint64_t)(s_gen[0] % kTailSlots) * T.partial_stride : base;
}

// `scratch` = shared memory the caller no longer needs: max(2*F*32, 512) doubles, 16-byte aligned.
template <int KIND>
__device__ __noinline__ void fold_tail(const TailParams& T, const void* partial, uint32_t q, uint32_t R, double* scratch,
                                       uint32_t seq, uint32_t dft_x) {
    __shared__ uint32_t s_prev;
    const uint32_t tid = threadIdx.x;
    const uint32_t p = blockIdx.x % q;
    const uint32_t slot = seq % kTailSlots;
    uint32_t* cnt = T.cnt + (size_t)slot * (q + 2u);
    constexpr uint32_t F = KIND == KIND_2BIT ? 64u : (KIND == KIND_I8 ? 16u : 4u);
    constexpr uint32_t E = F * 32u;

    __syncthreads();          // every thread's partial writes happen before thread 0's release below
    if (tid == 0) s_prev = arrive_acq_rel(cnt + p);
    __syncthreads();
    if (s_prev != R - 1u) return;

    // ---- stage A: replica sums of group p ---------------------------------------------------
    if (KIND == KIND_2BIT) {
        // thread t owns elements 8t .. 8t+7 (one 16-byte word of eight uint16 per replica)
        const uint4* src = reinterpret_cast<const uint4*>(partial) + (size_t)p * (E / 8u) + tid;
        const size_t stride = (size_t)q * (E / 8u);
        uint32_t a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        for (uint32_t r0 = 0; r0 < R; r0 += 8u) {
            uint4 v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = (r0 + k < R) ? __ldcg(src + (size_t)(r0 + k) * stride) : make_uint4(0, 0, 0, 0);
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                a[0] += v[k].x & 0xFFFFu; a[1] += v[k].x >> 16; a[2] += v[k].y & 0xFFFFu; a[3] += v[k].y >> 16;
                a[4] += v[k].z & 0xFFFFu; a[5] += v[k].z >> 16; a[6] += v[k].w & 0xFFFFu; a[7] += v[k].w >> 16;
            }
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint32_t e = 8u * tid + k, vslot = p * 32u + (e & 31u);
            const long long cnt = (long long)(T.cnt_quot + (vslot < T.cnt_rem ? 1u : 0u));
            scratch[e] = (double)(2ll * (long long)a[k] - 3ll * cnt);      // code sum -> level sum
        }
    } else {
        for (uint32_t e = tid; e < E; e += kThreads) {
            const size_t stride = (size_t)q * E;
            if (KIND == KIND_I8) {
                const int32_t* src = reinterpret_cast<const int32_t*>(partial) + (size_t)p * E + e;
                scratch[e] = (double)replica_sum<int32_t, long long>(src, stride, 0u, 1u, R);
            } else {
                const double* src = reinterpret_cast<const double*>(partial) + (size_t)p * E + e;
                scratch[e] = replica_sum<double, double>(src, stride, 0u, 1u, R);
            }
        }
    }
    __syncthreads();

    // ---- stage B: rotate, fold the group's W = 32*spv time samples into G[p] -----------------
    // B1: thread t multiplies the elements t, t+256, ... by their phasors -- all table loads of a thread
    //     in flight at once -- and leaves the products in shared memory (in place of the sums);
    // B2: tpp threads per (channel, bin) pair add the pair's products in a fixed order.
    const uint32_t n_bins = T.n_bins;      // (the parameters sit behind a reference: every use is a load -- the loops keep copies)
    const FastDiv dBins(n_bins), dC(T.C);  // (dividends below 2^24)
    const uint32_t pairs = T.C * n_bins, W = 32u * T.spv, tpp = T.tpp;
    const uint32_t base_b = dBins.mod(T.n0_mod_bins + p * W);
    {
        constexpr uint32_t EPT = (E + kThreads - 1) / kThreads;       // 8, 2, 1
        double v[EPT];
        double2 ph[EPT];
#pragma unroll
        for (uint32_t j = 0; j < EPT; ++j) {
            const uint32_t e = tid + j * kThreads;
            v[j] = 0.0; ph[j] = make_double2(1.0, 0.0);
            if (e < E) {
                const uint32_t f = e >> 5, ln = e & 31u;
                uint32_t t, c;
                dC.divmod(f, t, c);
                const uint32_t L = T.lut_len[c];
                v[j] = scratch[e];
                if (L > 1) ph[j] = __ldg(T.lut + T.lut_off[c] + (T.n0_mod_L[c] + p * W + ln * T.spv + t) % L);
            }
        }
        __syncthreads();
        double2* prod = reinterpret_cast<double2*>(scratch);
#pragma unroll
        for (uint32_t j = 0; j < EPT; ++j) {
            const uint32_t e = tid + j * kThreads;
            if (e < E) prod[e] = make_double2(v[j] * ph[j].x, v[j] * ph[j].y);
        }
        __syncthreads();
    }
    const double2* G = T.G + (size_t)slot * q * pairs;
    double2* Gp = T.G + ((size_t)slot * q + p) * pairs;
    {
        const uint32_t nC = T.C, spv_m1 = T.spv - 1u, spv_log2 = T.spv_log2, tpp_log2 = 31u - (uint32_t)__clz(tpp);   // tpp: a power of two
        const double2* prod = reinterpret_cast<const double2*>(scratch);
        const uint32_t dstep = tpp * n_bins, slots = pairs * tpp;
        for (uint32_t s0 = 0; s0 < slots; s0 += kThreads) {               // uniform trip count: shuffles below
            const uint32_t sl_ = s0 + tid;
            const bool active = sl_ < slots;
            const uint32_t pp = active ? sl_ >> tpp_log2 : 0u, u = sl_ & (tpp - 1u);
            uint32_t c, b;
            dBins.divmod(pp, c, b);
            double are = 0.0, aim = 0.0;
            if (active) {
                uint32_t d0 = b + n_bins - base_b; if (d0 >= n_bins) d0 -= n_bins;
                for (uint32_t d = d0 + u * n_bins; d < W; d += dstep) {
                    const double2 x = prod[(((d & spv_m1) * nC + c) << 5) + (d >> spv_log2)];
                    are += x.x; aim += x.y;
                }
            }
            for (uint32_t sh = tpp >> 1; sh > 0; sh >>= 1) {
                are += __shfl_xor_sync(0xFFFFFFFFu, are, sh);
                aim += __shfl_xor_sync(0xFFFFFFFFu, aim, sh);
            }
            if (active && u == 0) Gp[pp] = make_double2(are, aim);
        }
    }

    __syncthreads();
    if (tid == 0) s_prev = arrive_acq_rel(cnt + q);
    __syncthreads();
    // ---- stage C: groups in order, ragged tail, accumulate into the context ------------------
    // The last S group CTAs to arrive share it: the one that arrives as number q - S + k takes slice k of the (channel, bin)
    // pairs.  All but the very last wait (one thread, acquire loads) until every group has arrived -- the CTAs they wait for
    // are running -- so that a 16-channel stream is not finished by a single CTA.  Which CTA takes which slice changes
    // nothing in the arithmetic: every pair is summed by one thread in group order.
    const uint32_t S_want = (pairs + 127u) / 128u < kTailFinishers ? (pairs + 127u) / 128u : kTailFinishers;    // >= 128 pairs each
    const uint32_t S = q < S_want ? q : S_want;
    if (s_prev < q - S) return;
    const uint32_t slice = s_prev - (q - S);
    if (s_prev != q - 1u) {
        if (tid == 0) while (ld_acquire_u32(cnt + q) != q) __nanosleep(64);
        __syncthreads();
    }
    const uint32_t per_slice = (pairs + S - 1u) / S;
    const uint32_t pair_lo = slice * per_slice, pair_hi = pair_lo + per_slice < pairs ? pair_lo + per_slice : pairs;
    // The group sums and the ragged tail do not depend on P: they are formed first, and only then does the CTA wait
    // (first trip of the loop below) until P is up to date (n_done == seq) and no longer being read by a DFT kernel.
    auto wait_for_P = [&]() {
        if (tid == 0) {
            uint32_t a = ld_acquire_u32(&T.st->n_done), b = ld_acquire_u32(&T.st->dft_finished);
            while (a != seq || (int32_t)(b - dft_x) < 0) {
                __nanosleep(32);
                a = ld_acquire_u32(&T.st->n_done); b = ld_acquire_u32(&T.st->dft_finished);
            }
        }
        __syncthreads();
    };
    // thread = (slice sl of the groups, pair): slice sums first (all loads of a thread in flight at
    // once where possible), then the slices in order.
    const uint32_t my_pairs = pair_hi > pair_lo ? pair_hi - pair_lo : 0u;
    const uint32_t ppc = my_pairs < (uint32_t)kThreads ? (my_pairs ? my_pairs : 1u) : (uint32_t)kThreads;
    const uint32_t ns = (uint32_t)kThreads / ppc;            // >= 1; > 1 only when this CTA has fewer than 256 pairs
    const uint32_t sl = tid / ppc, e0 = tid % ppc;
    const uint32_t n_tail = (uint32_t)(T.n_total - T.NT);
    double* s_re = scratch;                                  // [kThreads]
    double* s_im = scratch + kThreads;                       // [kThreads]
    // A single finisher that OVERWRITES the bins and takes the DFT (one integration period per launch: pcal_integrate, series)
    // needs nothing from the earlier launches: it forms P and T first and only then waits for its turn to store them, so that
    // consecutive periods are serialised on a handful of stores instead of on the whole stage.  (<= 128 pairs: one trip below.)
    const bool early = S == 1u && T.overwrite && T.fuse_dft;
    bool waited = false;
    for (uint32_t pp0 = pair_lo; pp0 < pair_hi || !waited; pp0 += ppc) {        // uniform trip count; at least one trip (the wait)
        const uint32_t pp = pp0 + e0;
        double are = 0.0, aim = 0.0;
        if (sl < ns && pp < pair_hi) {
            for (uint32_t g0 = sl; g0 < q; g0 += 8u * ns) {
                double2 g[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) g[k] = (g0 + k * ns < q) ? __ldcg(G + (size_t)(g0 + k * ns) * pairs + pp) : make_double2(0.0, 0.0);
#pragma unroll
                for (int k = 0; k < 8; ++k) { are += g[k].x; aim += g[k].y; }
            }
        }
        if (ns > 1) {
            __syncthreads();
            s_re[tid] = are; s_im[tid] = aim;
            __syncthreads();
            are = 0.0; aim = 0.0;
            if (sl == 0) for (uint32_t k = 0; k < ns; ++k) { are += s_re[k * ppc + e0]; aim += s_im[k * ppc + e0]; }
        }
        const bool mine = sl == 0 && pp < pair_hi;
        uint32_t c = 0u, b = 0u;
        if (mine) dBins.divmod(pp, c, b);
        if (mine && n_tail) {   // samples NT .. n_total-1 (fewer than one vector)
            const uint32_t L = T.lut_len[c];
            const double2* lut = T.lut + T.lut_off[c];
            uint32_t bb = (uint32_t)((T.n0 + T.NT) % T.n_bins);
            uint32_t k = L > 1 ? (uint32_t)((T.n0 + T.NT) % L) : 0;
            for (uint32_t t = 0; t < n_tail; ++t) {
                if (bb == b) {
                    const double v = decode_tail(T.kind, T.sign_mag, T.tail, t, c, T.C);
                    if (L > 1) { const double2 ph = lut[k]; are += v * ph.x; aim += v * ph.y; }
                    else are += v;
                }
                if (++bb == T.n_bins) bb = 0;
                if (L > 1 && ++k == L) k = 0;
            }
        }
        if (early) {
            double2* sP = reinterpret_cast<double2*>(scratch + 2 * kThreads);
            if (mine) sP[pp] = make_double2(are, aim);
            __syncthreads();
            dft_in_cta(sP, sP + pairs, T.W, T.C, T.n_bins, T.dft_n1, T.k_shift % T.n_bins, nullptr, nullptr, kThreads, sP);
            wait_for_P(); waited = true;
            if (mine) {
                T.P[pp] = make_double2(are, aim);
                if (T.integer_exact) T.Pint[pp] = (long long)are;
                if (T.P_copy) T.P_copy[pp] = make_double2(are, aim);
                const double2 t = sP[pp];
                T.T_dev[pp] = t;
                if (T.T_host) T.T_host[pp] = t;
            }
            continue;
        }
        if (!waited) { wait_for_P(); waited = true; }        // every thread of the CTA, once
        if (!mine) continue;
        long long ai = (long long)are;     // exact: unrotated integer sums are integers below 2^53
        if (!T.overwrite) {
            const double2 cur = __ldcg(T.P + pp);          // L2: written by another SM under an overlapping grid
            are += cur.x; aim += cur.y;
            if (T.integer_exact) ai += __ldcg(T.Pint + pp);
        }
        T.P[pp] = make_double2(are, aim);
        if (T.integer_exact) T.Pint[pp] = ai;
        if (T.P_copy) T.P_copy[pp] = make_double2(are, aim);
        if (S == 1u && T.fuse_dft) reinterpret_cast<double2*>(scratch + 2 * kThreads)[pp] = make_double2(are, aim);   // (<= 128 pairs)
    }
    // the finishing CTAs meet once more; the last of them takes the DFT (pcal_integrate / series on small periods), makes the
    // slot ready for its next launch and publishes the result
    __syncthreads();
    if (S > 1u) {
        if (tid == 0) s_prev = arrive_acq_rel(cnt + q + 1u);
        __syncthreads();
        if (s_prev != S - 1u) return;
    }
    if (T.fuse_dft && !early) {   // T[c] = DFT(P[c]), every channel at once, from shared memory
        double2* sP = reinterpret_cast<double2*>(S > 1u ? scratch : scratch + 2 * kThreads);
        double2* sY = sP + pairs;
        if (S > 1u) {
            for (uint32_t pp = tid; pp < pairs; pp += kThreads) sP[pp] = __ldcg(T.P + pp);      // (slices written by the other finishers: L2)
            __syncthreads();
        }
        dft_in_cta(sP, sY, T.W, T.C, T.n_bins, T.dft_n1, T.k_shift % T.n_bins, T.T_dev, T.T_host, kThreads);
    }
    for (uint32_t i = tid; i <= q + 1u; i += kThreads) cnt[i] = 0u;    // ready for the slot's next launch
    __syncthreads();
    if (tid == 0) st_release_u32(&T.st->n_done, seq + 1u);             // P is final for this launch; the slot is free
}

}  // namespace pcal
