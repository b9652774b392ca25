// pcal_gen_mma.cuh -- generator path for int8 samples as a dense contraction on the tensor cores (eq. 2.3 + 2.2 with the
// phasor of eq. 2.5; BASELINE.json config 5).  (2-bit samples: pcal_gen2.cuh, the same algebra.)
//
// With the sample index written as n = n0 + 2^16 tile + 2048 row + pos (pos < 2048, row < 32),
//     P[b] = sum_{pos = b mod N_bins} e^{-j w pos} * sum_{tile,row} x[tile,row,pos] * rho[tile,row],
//     rho[tile,row] = e^{-j w (n0 + 2^16 tile)} * e^{-j w 2048 row}
// (the k-shift algebra of PAPER.md:97: the position factor is applied once at the end).  The inner sum is
// a matrix product  X^T (2048 positions x rows)  *  R (rows x digit columns)  -- a contraction over TIME.  It runs as
// integer tensor-core MMAs (mma.sync m16n8k16, s8 x s8 -> s32): the phasor is quantised to 31-bit fixed point,
// round(rho 2^30) = d0 + 2^8 d1 + 2^16 d2 + 2^24 d3 with signed 8-bit digits, and the eight digit columns (4 for Re,
// 4 for Im) fill the n = 8 side of the MMA.  All sums are exact integers (int32 per digit column; |sum| < 2^31 for the
// <= 256 tiles a CTA sees per launch), recombined and converted to fp64 once per launch.  The only approximation is the
// 2^-31 phasor quantisation (~5e-10 of a typical bin).
//
// Generator and resync.  rho[tile,row]: the tile factor comes from the exactly reduced INTEGER phase
// ((n0 + 2^16 tile) F_off mod F_s, the "fp64 phase resync every 2^16 samples" of BASELINE.json config 5),
// the row factor from a 32-entry table of exact stride phasors e^{-j w 2048 row} (stride stepping as in
// eq. 2.8); one coupled-form complex multiply (eq. 2.6) per row in fp64, never more than 31 strides from
// a resync point.  The 32 x 8 digit matrix of a tile is built by every warp for itself, lane = row.
//
// Data movement.  A row is 2048 positions (2048 B); warp w owns positions 256 w .. 256 w + 255 and thread
// (g = lane/4, t = lane%4) 32 of them for 8 of the 32 rows: the two 16-byte blocks c = 0, 1 at 256 w + 128 c + 16 g of rows
// 16h + 4t + j, loaded by the thread itself into its own cp.async ring (no barrier; a warp instruction covers 4 rows x
// 128 contiguous bytes).  The MMA wants four consecutive ROWS of one position in a register, memory has positions
// consecutive: a 4x4 byte transpose (8 PRMT per 16 bytes) turns 4 row words into 4 position words.  Rows past the end
// of the segment get zero digits, so whatever their ring slots hold contributes nothing.  ~1.2 instructions per sample
// instead of 3.75 for the FFMA2 kernel of pcal_gen.cuh: HBM-bound at any SM clock.
#pragma once
#include "pcal_gen.cuh"

namespace pcal {

constexpr uint32_t kMmaSpan = 2048;                    // positions per row
constexpr uint32_t kMmaRows = kTileSamples / kMmaSpan; // 32 rows per tile

template <int KIND> struct GenMmaCfg;
// LB bytes per load; GPT commit groups (of 4 loads: 4 consecutive rows) per tile; DG groups in flight per thread
template <> struct GenMmaCfg<KIND_I8>   { static constexpr int LB = 16, GPT = 4, DG = 4; };   // groups (h, block c)

template <int KIND>
constexpr size_t gen_mma_smem_bytes() {
    const size_t ring = (size_t)GenMmaCfg<KIND>::DG * 4 * kThreads * GenMmaCfg<KIND>::LB;
    const size_t fin = (size_t)kMmaSpan * sizeof(double2);              // final per-position values alias the ring
    return (size_t)kGenMaxTiles * sizeof(double2) + (kMmaRows + 128 + 16) * sizeof(double2) + (size_t)kWarps * 256 + (ring > fin ? ring : fin);
}

__device__ __forceinline__ void mma_s8_k16(int (&d)[4], uint32_t a0, uint32_t a1, uint32_t b0) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
                 : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
                 : "r"(a0), "r"(a1), "r"(b0));
}

// rows r0..r3 (bytes = 4 positions each) -> o[p] = (r0.p, r1.p, r2.p, r3.p), byte 0 = row 0
__device__ __forceinline__ void transpose4x4_bytes(uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3, uint32_t (&o)[4]) {
    const uint32_t x01l = __byte_perm(r0, r1, 0x5140), x01h = __byte_perm(r0, r1, 0x7362);
    const uint32_t x23l = __byte_perm(r2, r3, 0x5140), x23h = __byte_perm(r2, r3, 0x7362);
    o[0] = __byte_perm(x01l, x23l, 0x5410); o[1] = __byte_perm(x01l, x23l, 0x7632);
    o[2] = __byte_perm(x01h, x23h, 0x5410); o[3] = __byte_perm(x01h, x23h, 0x7632);
}

// signed base-256 digits of v (|v| <= 2^30): v = d0 + 2^8 d1 + 2^16 d2 + 2^24 d3; only their low bytes are used
__device__ __forceinline__ void digits4(int v, int& d0, int& d1, int& d2, int& d3) {
    d0 = v; v = (v + 128) >> 8;
    d1 = v; v = (v + 128) >> 8;
    d2 = v; d3 = (v + 128) >> 8;
}

template <int LB>
__device__ __forceinline__ void cp_async_pred(void* smem_dst, const void* gsrc, bool ok) {
    if (ok) cp_async_own<LB>(smem_dst, gsrc);
}

template <int KIND, bool SIGN_MAG>          // (KIND_I8, false: the only instantiation)
__global__ void __launch_bounds__(kThreads, 2) gen_mma_kernel(const __grid_constant__ GenParams P) {
    pdl_release();
    if (!P.input_ready) pdl_wait();
    constexpr int LB = GenMmaCfg<KIND>::LB, DG = GenMmaCfg<KIND>::DG;
    constexpr uint32_t ROW_BYTES = KIND == KIND_I8 ? kMmaSpan : kMmaSpan / 4;
    constexpr uint32_t TILE_BYTES = ROW_BYTES * kMmaRows;
    extern __shared__ __align__(16) unsigned char gen_smem[];
    double2* base = reinterpret_cast<double2*>(gen_smem);                       // [kGenMaxTiles] tile-start phasors
    double2* rtab = base + kGenMaxTiles;                                         // [32] exp(-j w 2048 row)
    double2* twA = rtab + kMmaRows;                                              // [128] exp(-j w 16 a): position factor, coarse part
    double2* twB = twA + 128;                                                    // [16]  exp(-j w b):    position factor, fine part
    unsigned char* bt_all = reinterpret_cast<unsigned char*>(twB + 16);          // [warp][8 digit columns][32 rows]
    unsigned char* ring = bt_all + kWarps * 256;                                 // [DG*4][kThreads][LB]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    unsigned char* bt = bt_all + warp * 256;

    const uint64_t n_rows = P.n_loads / (kMmaSpan / 16);                         // host loads = 16 samples; whole rows only (host guarantees a multiple)
    const uint32_t nt = blockIdx.x < P.n_tiles ? (uint32_t)((P.n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0;
    int acc[2][2][4][4];          // [block c][word half w2][byte b][C fragment]
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int w2 = 0; w2 < 2; ++w2)
#pragma unroll
            for (int b = 0; b < 4; ++b)
#pragma unroll
                for (int k = 0; k < 4; ++k) acc[c][w2][b][k] = 0;

    if constexpr (KIND == KIND_I8) {
    // this thread's loads of one tile, in consumption order: group-major, 4 consecutive rows per group
    //   l = 8h + 4c + j -> row 16h + 4t + j, block c
    constexpr int GPT = GenMmaCfg<KIND>::GPT;
    const unsigned char* gdata = reinterpret_cast<const unsigned char*>(P.data);
    const uint32_t col_off = (uint32_t)(warp * (ROW_BYTES / kWarps) + g * LB);
    // row (without the thread's 4t) and byte offset (without the thread's part) of load l: compile-time after unrolling
    auto row_c = [](int l) -> int { return KIND == KIND_I8 ? 16 * (l >> 3) + (l & 3) : 16 * (l >> 2) + (l & 3); };
    auto off_c = [&](int l) -> uint32_t {
        const uint32_t c = KIND == KIND_I8 ? (uint32_t)((l >> 2) & 1) : 0u;
        return (uint32_t)row_c(l) * ROW_BYTES + c * (ROW_BYTES / 16);
    };
    const uint32_t thread_off = (uint32_t)(4 * t) * ROW_BYTES + col_off;
    // ring slot of this thread inside its warp's 32*LB bytes: lanes that read consecutive global addresses
    // (same t, g = 0..7) sit in one contiguous run, so a cp.async of the warp writes whole shared-memory
    // lines; the run is permuted (g ^ 2t for 16-byte loads, g ^ 4(t/2) for 8-byte loads) so that every
    // LDS.128 quarter-warp / LDS.64 half-warp lands on distinct bank groups.
    const uint32_t chunk = (uint32_t)t * 8u + (LB == 16 ? (uint32_t)(g ^ (2 * t)) : (uint32_t)(g ^ (4 * (t >> 1))));
    unsigned char* my_ring = ring + ((size_t)warp * 32 + chunk) * LB;
    constexpr size_t SLOT = (size_t)kThreads * LB;
    const uint64_t tile_stride = (uint64_t)gridDim.x * TILE_BYTES;
    const long long row_stride = (long long)gridDim.x * kMmaRows;
    long long rows_left = (long long)n_rows - (long long)blockIdx.x * kMmaRows;  // rows from the start of this CTA's tile i on

    // issue the loads of commit group `grp` of a tile: src = the thread's first byte of that tile,
    // lim_t = (valid rows of that tile, 0..32) - 4t, so that load l is inside the data iff row_c(l) < lim_t
    auto issue_group = [&](const unsigned char* src, int lim_t, int grp, int slot_grp) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int l = grp * 4 + j;
            cp_async_pred<LB>(my_ring + (size_t)(slot_grp * 4 + j) * SLOT, src + off_c(l), row_c(l) < lim_t);
        }
        cp_async_commit();
    };
    auto lim_of = [&](long long left, bool exists) -> int {
        const int v = !exists || left <= 0 ? 0 : (left < (long long)kMmaRows ? (int)left : (int)kMmaRows);
        return v - 4 * t;
    };
    // prologue: DG groups = DG/GPT tiles ahead
    static_assert(DG % GPT == 0, "whole tiles in flight");
    constexpr uint32_t TA = DG / GPT;
    const unsigned char* ahead = gdata + (uint64_t)blockIdx.x * TILE_BYTES + thread_off;   // tile i + TA after the prologue
    long long ahead_left = rows_left;
#pragma unroll
    for (uint32_t ti = 0; ti < TA; ++ti) {
        const int lim_t = lim_of(ahead_left, ti < nt);
#pragma unroll
        for (int gq = 0; gq < GPT; ++gq) issue_group(ahead, lim_t, gq, (int)(ti * GPT + gq));
        ahead += tile_stride; ahead_left -= row_stride;
    }

    // (the first loads are in flight: now the tables)
    {   // resync table: the exactly reduced integer phase of every tile start of this CTA -> fp64 phasor
        uint64_t k_cta = P.k0 + mulmod_u64(P.E, blockIdx.x, P.Fs);
        if (k_cta >= P.Fs) k_cta -= P.Fs;
        for (uint32_t i = tid; i < nt; i += kThreads) {
            uint64_t k = k_cta + mulmod_u64(P.D, i, P.Fs);
            if (k >= P.Fs) k -= P.Fs;
            base[i] = phasor_neg(k, P.Fs);
        }
        // (the last 32 threads: the first ones are busy with the tile phasors above)
        if (tid >= kThreads - (int)kMmaRows) { const int r = tid - (kThreads - (int)kMmaRows); rtab[r] = phasor_neg(mulmod_u64(P.Foff, (uint64_t)r * kMmaSpan, P.Fs), P.Fs); }
        // position factors exp(-j w pos), pos = 16 a + b, for the epilogue: threads 64 .. 207, exactly reduced as well
        if (tid >= 64 && tid < 64 + 128) twA[tid - 64] = phasor_neg(mulmod_u64(P.Foff, (uint64_t)(tid - 64) * 16u, P.Fs), P.Fs);
        if (tid >= 192 && tid < 192 + 16) twB[tid - 192] = phasor_neg(mulmod_u64(P.Foff, (uint64_t)(tid - 192), P.Fs), P.Fs);
    }
    __syncthreads();

    for (uint32_t i = 0; i < nt; ++i, rows_left -= row_stride, ahead += tile_stride, ahead_left -= row_stride) {
        const int ahead_lim_t = lim_of(ahead_left, i + TA < nt);
        // ---- digit matrix of this tile: lane = row ----
        {
            const double2 b0 = base[i], r = rtab[lane];
            const bool valid = (long long)lane < rows_left;
            const int vre = valid ? __double2int_rn((b0.x * r.x - b0.y * r.y) * 1073741824.0) : 0;
            const int vim = valid ? __double2int_rn((b0.x * r.y + b0.y * r.x) * 1073741824.0) : 0;
            int d0, d1, d2, d3, e0, e1, e2, e3;
            digits4(vre, d0, d1, d2, d3); digits4(vim, e0, e1, e2, e3);
            __syncwarp();             // every lane is done with the previous tile's digits
            bt[0 * 32 + lane] = (unsigned char)d0; bt[1 * 32 + lane] = (unsigned char)d1; bt[2 * 32 + lane] = (unsigned char)d2;
            bt[3 * 32 + lane] = (unsigned char)d3; bt[4 * 32 + lane] = (unsigned char)e0; bt[5 * 32 + lane] = (unsigned char)e1;
            bt[6 * 32 + lane] = (unsigned char)e2; bt[7 * 32 + lane] = (unsigned char)e3;
            __syncwarp();
        }
        const uint32_t* bt32 = reinterpret_cast<const uint32_t*>(bt);
        const uint32_t bf[2] = {bt32[g * 8 + t], bt32[g * 8 + 4 + t]};        // rows 4t.., 16+4t.. of digit column g

#pragma unroll
        for (int grp = 0; grp < GPT; ++grp) {
            const int h = KIND == KIND_I8 ? (grp >> 1) : grp;
            const int slot_grp = (int)((i * (uint32_t)GPT + grp) % DG);
            cp_async_wait<DG - 1>();
            auto refill = [&]() { issue_group(ahead, ahead_lim_t, grp, slot_grp); };   // the slot group just read: same group, TA tiles ahead
            if constexpr (KIND == KIND_I8) {
                const int c = grp & 1;
                uint32_t T[4][4];     // [word][byte]: 4 rows of one position
                uint4 v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] = *reinterpret_cast<const uint4*>(my_ring + (size_t)(slot_grp * 4 + j) * SLOT);
#pragma unroll
                for (int w = 0; w < 4; ++w) transpose4x4_bytes(word_of(v[0], w), word_of(v[1], w), word_of(v[2], w), word_of(v[3], w), T[w]);
                refill();
#pragma unroll
                for (int w2 = 0; w2 < 2; ++w2)
#pragma unroll
                    for (int b = 0; b < 4; ++b) mma_s8_k16(acc[c][w2][b], T[w2][b], T[w2 + 2][b], bf[h]);
            }
        }
    }
    }
    cp_async_wait<0>();
    __syncthreads();                  // the ring is free: it becomes the per-position result array

    // ---- digits -> fp64, post-twiddle by exp(-j w pos), positions -> bins ------------------------
    // The three Re and three Im digit sums of a position sit in lanes t = 0, 1, 2 of a quad: every thread leaves its 64
    // int32 sums in shared memory ([element][thread]: conflict-free), then lane t of the quad finishes the positions
    // idx % 4 == t of its quad (eight each), all reads before the result array -- which aliases the dump -- is written.
    int* dump = reinterpret_cast<int*>(ring);               // [64][kThreads]
    double* pos_re = reinterpret_cast<double*>(ring);      // [2048]
    double* pos_im = pos_re + kMmaSpan;
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int w2 = 0; w2 < 2; ++w2)
#pragma unroll
            for (int b = 0; b < 4; ++b)
#pragma unroll
                for (int k = 0; k < 4; ++k) dump[((((c * 2 + w2) * 4 + b) * 4) + k) * kThreads + tid] = acc[c][w2][b][k];
    __syncthreads();
    long long fre[8], fim[8];
    {
        const int qb = tid & ~3;                            // lane 0 of this thread's quad
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            const int idx = 4 * m + t;                      // ((c*2 + w2)*4 + b)*2 + half
            const int half = idx & 1, e0 = (idx >> 1) * 4 + 2 * half;      // elements e0, e0+1 = C-fragment columns 2t', 2t'+1
            // digit columns: lane 0 holds (Re0, Re1), lane 1 (Re2, Re3), lane 2 (Im0, Im1), lane 3 (Im2, Im3)
            const long long r0 = dump[e0 * kThreads + qb], r1 = dump[(e0 + 1) * kThreads + qb];
            const long long r2 = dump[e0 * kThreads + qb + 1], r3 = dump[(e0 + 1) * kThreads + qb + 1];
            const long long i0 = dump[e0 * kThreads + qb + 2], i1 = dump[(e0 + 1) * kThreads + qb + 2];
            const long long i2 = dump[e0 * kThreads + qb + 3], i3 = dump[(e0 + 1) * kThreads + qb + 3];
            fre[m] = r0 + 256 * r1 + 65536 * r2 + 16777216 * r3;
            fim[m] = i0 + 256 * i1 + 65536 * i2 + 16777216 * i3;
        }
    }
    __syncthreads();                                        // the dump has been read: the result array may overwrite it
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        const int idx = 4 * m + t, half = idx & 1, b = (idx >> 1) & 3, w2 = (idx >> 3) & 1, c = idx >> 4;
        const int wsel = w2 + 2 * half;                     // word of the block
        const uint32_t pos = (uint32_t)(warp * 256 + c * 128 + g * 16 + 4 * wsel + b);
        const long long pre = fre[m], pim = fim[m];
        pos_re[pos] = (double)pre * (1.0 / 1073741824.0);
        pos_im[pos] = (double)pim * (1.0 / 1073741824.0);
    }
    __syncthreads();
    {   // exp(-j w pos), pos = tid + 256 k = 16 a + b: product of two exactly reduced table phasors (built in the prologue)
        const double2 fb = twB[tid & 15];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const double2 fa = twA[(tid >> 4) + 16 * k];
            const double twx = fa.x * fb.x - fa.y * fb.y, twy = fa.x * fb.y + fa.y * fb.x;
            const uint32_t pos = (uint32_t)tid + 256u * k;
            const double re = pos_re[pos], im = pos_im[pos];
            pos_re[pos] = re * twx - im * twy;
            pos_im[pos] = re * twy + im * twx;
        }
    }
    __syncthreads();
    pdl_wait();   // the partial bins of the previous launch may still be read by its post kernel
    for (uint32_t sb = tid; sb < P.n_bins; sb += kThreads) {
        double re = 0.0, im = 0.0;
        for (uint32_t pos = sb; pos < kMmaSpan; pos += P.n_bins) { re += pos_re[pos]; im += pos_im[pos]; }
        P.tail.partial[(size_t)blockIdx.x * P.n_bins + sb] = make_double2(re, im);
    }
}

}  // namespace pcal
