// pcal_gen_tail.cuh -- the reduction behind the generator kernels of pcal_gen.cuh / pcal_gen_mma.cuh, run INSIDE them by the
// CTA that finishes last (a5 of SURVEY section 8: "the step the paper leaves to the host CPU"):
// per-CTA partial bins -> bins (CTA order, fixed: the tile assignment of these kernels is static), ragged tail with exactly
// reduced phases, accumulation into the context and, for pcal_integrate / pcal_extract_series, the DFT.
// A generator step is thereby ONE launch.  Launches overlap like the fold kernels do (pcal_tail.cuh, "Pipelining"): partials
// and arrival counters live in a ring of kTailSlots slots, every CTA takes a ticket before its dependent grid may start, and
// the three ordering conditions of the TailState replace the grid-wide wait.
#pragma once
#include "pcal_tail.cuh"

namespace pcal {

struct GenTailParams {
    TailState* st;            // [device] tickets and progress counters of the context
    uint32_t* cnt;            // [device] [slot][2] arrival counters (grid, finishers), zero between launches
    double2* partial;         // [device] [slot][grid][n_bins] per-CTA partial bins, bin index relative to the piece start
    double2* P;               // [device] folded bins [n_bins]
    const uint8_t* tail;      // [device] first byte after the last sample the CTAs have served
    uint64_t n0, n_body, n_total;   // absolute index of the first sample; samples served by the CTAs; samples in the piece
    uint64_t Fs, Foff;
    uint32_t n_bins;
    int kind, sign_mag, overwrite;
    int fuse_dft;             // 1: the last CTA also takes the DFT in two stages (dft_in_cta), N_bins = dft_n1 * N2
    uint32_t dft_n1, k_shift;
    const double2* W;         // [device] exp(-j 2 pi k / N_bins)
    double2 *T_dev, *T_host, *P_copy;
};

// One thread (the caller picks it) takes the launch's ticket: s_gen[0] = sequence number, s_gen[1] = dft_started seen.  It
// returns once the slot's previous user (launch seq - kTailSlots) has finished.  The caller's next barrier publishes s_gen;
// only after it may the CTA release its dependent grid.
__device__ __forceinline__ void gen_take_ticket(const GenTailParams& T, uint32_t* s_gen) {
    const unsigned long long tk = atomicAdd(&T.st->tick, 1ull);       // (ticket and acquire load in flight together: pcal_tail.cuh)
    uint32_t done, x;
    ld_acquire_done_started(T.st, done, x);
    const uint32_t seq = (uint32_t)(tk / gridDim.x);
    s_gen[0] = seq; s_gen[1] = x;
    if ((int32_t)(done - (seq - kTailSlots + 1u)) < 0)
        while ((int32_t)(ld_acquire_u32(&T.st->n_done) - (seq - kTailSlots + 1u)) < 0) __nanosleep(64);
}

__device__ __forceinline__ double2* gen_partial_of(const GenTailParams& T, const uint32_t* s_gen) {
    return T.partial + ((size_t)(s_gen[0] % kTailSlots) * gridDim.x + blockIdx.x) * T.n_bins;
}

// Called by every thread of the CTA (256 threads) after it has written its partial bins.  `scratch`: shared memory the
// caller no longer needs, 16-byte aligned, at least (2 * n_bins + 512) double2 when fuse_dft, else (n_bins + 512).
// The last S CTAs to arrive share the work (S = 1..8, one per 16384 partial values): the one that arrives as number
// grid - S + k sums slice k of the bins over every CTA; all but the very last wait for the rest with acquire loads (the CTAs
// they wait for are running or queued behind launches that finish on their own).  Which CTA takes which slice changes
// nothing in the arithmetic.
__device__ __forceinline__ void gen_tail(const GenTailParams& T, uint32_t* s_gen, double2* scratch) {
    const uint32_t tid = threadIdx.x, lane = tid & 31u, sl = tid >> 5;
    const uint32_t seq = s_gen[0], slot = seq % kTailSlots, dft_x = s_gen[1];
    uint32_t* cnt = T.cnt + 2u * slot;
    __syncthreads();          // every thread's partial writes happen before thread 0's release below
    if (tid == 0) s_gen[3] = arrive_acq_rel(cnt);
    __syncthreads();
    const uint32_t want = (uint32_t)(((uint64_t)gridDim.x * T.n_bins + 16383u) / 16384u);
    const uint32_t S = want < 1u ? 1u : (want > kTailFinishers ? kTailFinishers : want);
    const uint32_t arrived = s_gen[3];
    if (arrived < gridDim.x - S) return;
    const uint32_t slice = arrived - (gridDim.x - S);
    if (arrived != gridDim.x - 1u) {
        if (tid == 0) while (ld_acquire_u32(cnt) != gridDim.x) __nanosleep(64);
        __syncthreads();
    }
    uint32_t per = (T.n_bins + S - 1u) / S;
    per = (per + 31u) & ~31u;                                // whole groups of 32 bins
    const uint32_t bin_lo = slice * per < T.n_bins ? slice * per : T.n_bins;
    const uint32_t bin_hi = bin_lo + per < T.n_bins ? bin_lo + per : T.n_bins;

    // ---- partial bins of every CTA in CTA order (eight slices of CTAs, then the slices in order) ----
    uint32_t seen_done = 0, seen_dft = 0;
    if (tid == 0) { seen_done = ld_acquire_u32(&T.st->n_done); seen_dft = ld_acquire_u32(&T.st->dft_finished); }
    const double2* part = T.partial + (size_t)slot * gridDim.x * T.n_bins;
    double2* sP = scratch;                                   // [n_bins] the piece's bins, then the accumulated bins
    double2* red = scratch + T.n_bins;                       // [8][32] slice sums (then, with fuse_dft, [n_bins] DFT scratch)
    const uint32_t shift = (uint32_t)(T.n0 % T.n_bins);
    const uint32_t n_tail = (uint32_t)(T.n_total - T.n_body);
    for (uint32_t b0 = bin_lo; b0 < bin_hi; b0 += 32u) {     // uniform trip count
        const uint32_t b = b0 + lane;
        const bool ok = b < bin_hi;
        uint32_t s = ok ? b + T.n_bins - shift : 0u; if (s >= T.n_bins) s -= T.n_bins;
        double re = 0.0, im = 0.0;
        if (ok) {
            for (uint32_t c0 = sl; c0 < gridDim.x; c0 += 64u) {        // eight loads in flight, added in CTA order
                double2 v[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = (c0 + 8u * k < gridDim.x) ? __ldcg(part + (size_t)(c0 + 8u * k) * T.n_bins + s) : make_double2(0.0, 0.0);
#pragma unroll
                for (int k = 0; k < 8; ++k) { re += v[k].x; im += v[k].y; }
            }
        }
        red[tid] = make_double2(re, im);
        __syncthreads();
        if (sl == 0 && ok) {
            re = 0.0; im = 0.0;
#pragma unroll
            for (int ww = 0; ww < 8; ++ww) { re += red[ww * 32 + lane].x; im += red[ww * 32 + lane].y; }
            if (n_tail) {     // samples n_body .. n_total-1 of this bin, in order, exactly reduced phases
                const uint32_t bb0 = (uint32_t)((T.n0 + T.n_body) % T.n_bins);
                for (uint32_t t = (b + T.n_bins - bb0) % T.n_bins; t < n_tail; t += T.n_bins) {
                    const double v = decode_tail(T.kind, T.sign_mag, T.tail, t, 0, 1);
                    const double2 ph = phasor_neg(mulmod_u64(T.Foff, T.n0 + T.n_body + t, T.Fs), T.Fs);
                    re += v * ph.x; im += v * ph.y;
                }
            }
            sP[b] = make_double2(re, im);
        }
        __syncthreads();
    }
    // P of every earlier launch must be in place (n_done == seq) and no earlier DFT kernel may still be reading it
    if (tid == 0) {
        uint32_t a = seen_done, b = seen_dft;
        while (a != seq || (int32_t)(b - dft_x) < 0) {
            __nanosleep(32);
            a = ld_acquire_u32(&T.st->n_done); b = ld_acquire_u32(&T.st->dft_finished);
        }
    }
    __syncthreads();
    for (uint32_t b = bin_lo + tid; b < bin_hi; b += blockDim.x) {
        double2 v = sP[b];
        if (!T.overwrite) { const double2 cur = __ldcg(T.P + b); v.x += cur.x; v.y += cur.y; }
        T.P[b] = v;
        sP[b] = v;
        if (T.P_copy) T.P_copy[b] = v;
    }
    __syncthreads();
    if (S > 1u) {             // the finishers meet once more; the last of them goes on
        if (tid == 0) s_gen[3] = arrive_acq_rel(cnt + 1);
        __syncthreads();
        if (s_gen[3] != S - 1u) return;
        if (T.fuse_dft) {
            for (uint32_t b = tid; b < T.n_bins; b += blockDim.x) sP[b] = __ldcg(T.P + b);     // (slices written by the other finishers: L2)
            __syncthreads();
        }
    }
    if (T.fuse_dft) dft_in_cta(sP, red, T.W, 1u, T.n_bins, T.dft_n1, T.k_shift % T.n_bins, T.T_dev, T.T_host, blockDim.x);
    if (tid == 0) { cnt[0] = 0u; cnt[1] = 0u; }                        // ready for the slot's next launch
    __syncthreads();
    if (tid == 0) st_release_u32(&T.st->n_done, seq + 1u);             // P is final for this launch; the slot is free
}

}  // namespace pcal
