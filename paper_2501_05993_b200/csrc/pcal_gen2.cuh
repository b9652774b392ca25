// pcal_gen2.cuh -- generator path for 2-bit samples (1, 2 or 4 channels per word group): eq. 2.3 + 2.2 with the
// phasor of eq. 2.5 as a dense contraction over TIME on the tensor cores, one launch per piece.
//
// Algebra (as in pcal_gen_mma.cuh, the int8 kernel).  A piece is cut into ROWS of span_t time samples; span_t is a multiple
// of N_bins and of the samples per 16 bytes, so a field position keeps its bin from row to row.  With
// n = n0 + span_t R + tau (R = row, tau < span_t),
//     P_c[b] = sum_{tau = b - n0 mod N_bins} e^{-j w_c tau} * sum_R x_c[R, tau] * rho_c[R],     rho_c[R] = e^{-j w_c (n0 + span_t R)}
// (the k-shift algebra of PAPER.md:97: the position factor is applied once at the end).  The inner sum is the matrix
// product X^T (positions x rows) * R (rows x digit columns): mma.sync m16n8k32 u8 x s8 -> s32 with the phasor quantised
// to 31-bit fixed point, round(rho 2^30) = d0 + 2^8 d1 + 2^16 d2 + 2^24 d3 (signed 8-bit digits; 4 Re + 4 Im columns =
// the n = 8 side of the MMA).  Every sum is an exact integer; the only approximation is the 2^-31 phasor quantisation
// (~5e-10 of a typical bin).
// Rows are SHORT (span_t = the smallest admissible multiple with at least 8 sixteen-byte chunks; config 3: 512 samples
// = N_bins): few positions mean few accumulators (16 registers per thread instead of 64), a small epilogue and a small
// cross-CTA reduction, at the price of more phasors (one per row).
//
// Generator and resync (eq. 2.5-2.8).  rho_c[R] = base0 * hi[B / 256] * lo[B % 256] * row[r] for row r of batch B (a batch
// = 4 tiles = 512 rows at most, <= 2^18 samples): four table phasors, each evaluated in long double on the host from an
// exactly reduced INTEGER phase, three coupled-form multiplies (eq. 2.6) deep in fp64.  Nothing is carried from batch to
// batch or from row to row -- every row restarts from the tables ("fp64 phase resync", BASELINE.json config 5, at every
// row) -- so there is no drift to bound; the error of rho is ~4e-16 before the 2^-31 quantisation.
//
// Structure (profiles/r2_ncu_full.md has the before/after against the round-1 kernel):
//   * warp roles, no CTA-wide barrier in the loop.  Warps 1..3 (generators) write the digit matrices of the CTA's tile
//     sequence -- its own batches first, then batches that warp 1 claims from a device counter, each claim issued two
//     batches ahead -- into a ring of entries, taking the tiles of the sequence in turn.  Their latency per tile is the
//     critical resource of the kernel (one warp: 0.86 of the copy peak on config 3, two: 0.92, three: 0.97): row phasors
//     of a batch in shared memory, digits by one fp64 add and one xor (g2_item_digits).  Warp 0 (loader) follows the
//     sequence and copies each tile as it lies in memory (one cp.async instruction per 512 contiguous bytes) into a ring
//     of padded tiles; completion arrives on the stage's mbarrier (cp.async.mbarrier.arrive.noinc).  Warps 4..11
//     (consumers) wait for "full", read their operands and release stage and digit entry on "empty" barriers.  Nobody
//     waits for anybody else's loads.
//   * the 4x4 byte transpose (four rows of one position into one register) is done by the load itself:
//     ldmatrix.m16n16.trans.b8 (SASS LDSM.8.MT1616, new on sm_100) returns exactly the A fragment of m16n8k32, lane
//     (g, t): byte column g / g + 8 of rows 4t..4t+3 (+16).  The row pitch is an odd number of 16-byte chunks, which keeps
//     it conflict-free.  No PRMT.
//   * the four 2-bit fields of a byte are separated by PREFIX masks: U0 = byte, U1 = byte & 0xFC, U2 = & 0xF0,
//     U3 = & 0xC0 (3 LOP3 instead of 4; single channel), the field sums S_f are differences of the U sums, exact.
//     With C = 2 / 4 channels field f belongs to channel f mod C and is masked accordingly (digits per channel).
//   * hybrid tile assignment: three quarters of the batches are a CTA's own (index + k * grid), the rest are claimed from a
//     device counter -- a CTA that starts late simply takes fewer.  A CTA is half an SM (384 threads, 80 registers) and
//     lets its dependent grid start as soon as its ticket is taken: consecutive launches share the SMs pairwise and HBM
//     keeps streaming while one of them is in its epilogue.
//   * the per-position sums of a CTA are exact int64 and are added to the launch's accumulators with integer
//     red.global.add -- associative, so the result is bit-identical whatever the tile assignment was.  The CTA that
//     arrives last converts to fp64, applies the position factor, folds positions to bins in a fixed order, adds the
//     ragged tail and accumulates into the context (same TailState protocol as pcal_tail.cuh) and, for pcal_integrate /
//     pcal_extract_series, takes the DFT in two stages (dft_in_cta).
//   * words of 8 / 16 channels: a time sample is 2 / 4 bytes ("classes" of four channels).  An MMA's 16 byte columns hold every
//     class while its digit matrix belongs to one channel: the masked operand meets the digits of channel u of every class in turn
//     (NCLS MMAs), each lane keeps the sums of its own class.  All classes in one launch when the accumulators fit (rows of <= 16
//     chunks: NCLS = 2 or 4, one CTA per SM), else one class per launch.  Rows longer than 2048 fields: column blocks of 32
//     chunks, one launch each.
#pragma once
#include "pcal_gen.cuh"
#include "pcal_tail.cuh"

namespace pcal {

constexpr int kG2Consumers = 8;                               // consumer warps
constexpr int kG2Threads = (kG2Consumers + 4) * 32;           // + loader + at most three generator warps
constexpr uint32_t kG2StageBytes = 18432;                     // a padded tile: 128 rows x 144 B (8 chunks) ... 32 rows x 528 B (32 chunks)
constexpr uint32_t kG2Fields = 2048;                          // fields (positions) per row at most
constexpr uint32_t kG2Batch = 4;                              // tiles per claim
constexpr uint32_t kG2CapBatches = 256;                       // claims per CTA per launch: <= 1032 tiles keep the int32 digit sums exact
constexpr uint32_t kG2MaxCh = 16;                             // channels per launch at most (four per byte class, four classes)
constexpr uint32_t kG2Invalid = 0xFFFFFFFFu;
constexpr uint32_t kG2DigRG = 72;                             // words of a digit matrix (one channel, one group of 32 rows): 64 + 8 of padding
constexpr uint32_t kG2TabRows = 512, kG2TabLo = 256, kG2TabHi = 128;      // generator tables per channel: rows of a batch, lo, hi
constexpr uint32_t kG2TabStride = kG2TabRows + kG2TabLo + kG2TabHi;

// Shared memory of a CTA (two CTAs share an SM): ring of sample tiles | ring of digit matrices (the generator runs that far
// ahead of the consumers) | the generator's row table of one batch (4 tiles; when it fits) | barriers and bookkeeping
constexpr size_t kG2SmemBudget = 115712 - 256;                // (228 KB - 2 x 1 KB reserved) / 2, less the kernel's static variables
constexpr size_t kG2SmemBudgetAlone = 232448 - 1024;          // one CTA per SM (several byte classes per launch: the accumulators need the registers)
// C = channels per byte (1, 2, 4); NCLS = byte classes served by one launch (words of 8 / 16 channels: a time sample is 2 / 4 bytes,
// "classes"; else 1); CPW = chunks per consumer warp
template <int C, int CPW, int NCLS> struct G2Cfg {
    static constexpr int CT = C * NCLS;                                        // channels of a launch
    static constexpr int KG = 4 / CPW, RT = 32 * KG;                          // row groups (K = 32 rows each) and rows per tile
    static constexpr int DIGITS = 8;   // digit entries: how far the generators run ahead
    // generator work items per tile and lane: (channel, row quad) pairs / 32.  Three generator warps take the tiles of the
    // CTA's sequence in turn.  With more than 32 items LC = 32 / CT lanes share a channel; the per-channel strides of the
    // digit matrices and of the row table are padded by LC words / entries, which spreads the lanes of a warp over the banks.
    static constexpr int KI = (CT * RT / 4 + 31) / 32, NG = 3, THREADS = (kG2Consumers + 1 + NG) * 32;
    static constexpr int LC = CT * RT / 4 <= 32 ? RT / 4 : 32 / CT;                                // lanes per channel
    static constexpr int DIG_CH = KG * (int)kG2DigRG + (KI > 1 ? LC : 0);     // words of a channel's digit matrices [KG][8 columns][8 quads] (+ pad)
    static constexpr uint32_t DIG_BYTES = (uint32_t)CT * DIG_CH * 4;          // digit matrices of a tile
    static constexpr int TAB_CH = 4 * RT + (KI > 1 && LC < 8 ? LC : 0);       // entries of a channel's row table (+ pad)
    static constexpr uint32_t TAB_BYTES = (uint32_t)CT * TAB_CH * 16;         // exp(-j w_c span_t r), r < rows of a batch
    static constexpr size_t FIXED = (size_t)DIGITS * DIG_BYTES + 1024;
    static constexpr size_t BUDGET = NCLS == 1 ? kG2SmemBudget : kG2SmemBudgetAlone;
    static constexpr int MAXT = NCLS == 1 ? 5 : 8;                            // (alone on the SM: a deeper ring keeps as many bytes in flight as two CTAs would)
    static constexpr bool TAB_SMEM = 4 * (size_t)kG2StageBytes + FIXED + TAB_BYTES <= BUDGET;
    static constexpr size_t ROOM = BUDGET - FIXED - (TAB_SMEM ? TAB_BYTES : 0u);
    static constexpr int TILES = ROOM / kG2StageBytes >= (size_t)MAXT ? MAXT : (int)(ROOM / kG2StageBytes);
    static constexpr size_t BYTES = (size_t)TILES * kG2StageBytes + FIXED + (TAB_SMEM ? TAB_BYTES : 0u);
};

struct Gen2Params {
    const unsigned char* data;     // [device] packed samples of this piece, 16-byte aligned
    uint64_t n_rows;               // complete rows in the piece
    uint32_t n_tiles, n_batches;   // ceil(n_rows / rows per tile), ceil(n_tiles / kG2Batch)
    uint32_t n_static;             // batches every CTA takes without asking (>= 1): about 3/4 of the launch
    uint32_t chunks, row_bytes;    // 16-byte chunks of a row that this launch serves (<= 32), 16 * chunks
    uint64_t row_stride, col_off;  // bytes from row to row in memory; first byte of this launch's columns in a row (rows longer than 32
                                   // chunks are served in column blocks, one launch each; else row_bytes, 0)
    uint32_t tau0;                 // time offset of the first position of this launch's columns inside a row
    int do_tail;                   // this launch also adds the ragged tail of the piece
    uint32_t pitch;                // row pitch in shared memory: row_bytes (+16 if chunks is even)
    uint32_t span_t;               // time samples per row (multiple of N_bins)
    uint32_t cls_count, cls;       // words of 8 / 16 channels: a time sample is cls_count bytes ("classes"), this launch serves bytes
                                   // cls .. cls + NCLS - 1 of each (channels 4 cls ..; the other bytes' sums are not used); else 1, 0
    uint32_t c_real, c_base;       // channels in the stream; first channel of this launch
    uint64_t Fs;
    uint64_t Foff[kG2MaxCh];       // rotator frequency per channel (micro-hertz, k-shift included): ragged tail
    double2 base0[kG2MaxCh];       // exp(-j w_c n0): phasor of the first sample of the piece (exactly reduced phase, long double on the host)
    const double2* gtab;           // [device] [C][kG2TabStride] generator tables, each entry from an exactly reduced phase in long double:
                                   //   [0..511] exp(-j w_c span_t r) rows of a batch; [512..767] exp(-j w_c D k), D = samples per batch;
                                   //   [768..895] exp(-j w_c 256 D k)
    const double2* tw;             // [device] [C][span_t] exp(-j w_c tau)
    uint32_t* ctr;                 // [device] [slot][2]: batch counter, arrival counter; zero between launches
    long long* posacc;             // [device] [slot][2 * kG2Fields] exact per-position sums (re, im) * 2^30; zero between launches
    TailState* st;                 // [device] tickets and progress counters of the context
    // final stage
    double2* P;                    // [device] folded bins [C][N_bins]
    const uint8_t* tail;           // [device] first byte after the last complete row
    uint64_t n0, n_body, n_total;  // absolute index of the first sample; samples in complete rows; samples in the piece
    uint32_t n_bins, n0_mod_bins;
    int overwrite, input_ready;
    int fuse_dft;                  // 1: the last CTA also takes the DFT, two stages N_bins = dft_n1 * N2 (pcal_post.cuh)
    uint32_t dft_n1;
    uint32_t k_shift;
    const double2* W;              // [device] exp(-j 2 pi k / N_bins)
    double2 *T_dev, *T_host, *P_copy;
};

template <int C, int CPW, int NCLS>
constexpr size_t gen2_smem_bytes() {
    return G2Cfg<C, CPW, NCLS>::BYTES;
}

// ---- mbarrier / cp.async / ldmatrix helpers -----------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "G2_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra G2_DONE;\n"
        "bra G2_WAIT;\n"
        "G2_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// the arrival happens when every cp.async this thread issued before has landed; counted in the barrier's init count
__device__ __forceinline__ void cp_async_arrive_noinc(uint32_t bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
// 16 bytes global -> shared (SASS LDGSTS.E.BYPASS.128), offsets as immediates where they are compile-time constants
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
template <uint32_t DOFF, uint32_t SOFF>
__device__ __forceinline__ void cp_async16_imm(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0 + %2], [%1 + %3], 16;" ::"r"(dst), "l"(src), "n"(DOFF), "n"(SOFF) : "memory");
}
// warp loads K0..K1-1 of a complete tile: load k covers the 512 contiguous bytes k*512.. of the tile; in shared memory they
// are DSTEP bytes apart (512 bytes = a whole number of rows for 8, 16 or 32 chunks per row)
template <uint32_t K0, uint32_t K1, uint32_t DSTEP>
__device__ __forceinline__ void g2_copy_tile(uint32_t dst, const void* src) {
    if constexpr (K0 < K1) {
        cp_async16_imm<K0 * DSTEP, K0 * 512u>(dst, src);
        g2_copy_tile<K0 + 1, K1, DSTEP>(dst, src);
    }
}
// two 16 x 16 byte matrices, transposed: lanes 0..15 give the rows of the first, 16..31 of the second.  Lane (g, t)
// receives r0 = byte column g of rows 4t..4t+3, r1 = byte column g + 8, r2 / r3 the same of the second matrix:
// the A fragment of mma.m16n8k32 with M = byte column and K = row.
__device__ __forceinline__ void ldsm_t8_x2(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m16n16.x2.trans.shared.b8 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr) : "memory");
}
__device__ __forceinline__ void mma_u8s8_k32(int (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void red_add_s64(long long* p, long long v) {
    asm volatile("red.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// prefix / channel masks of the four "combinations" u = 0..3 of a byte and the channel whose digits they meet
template <int C> __device__ __forceinline__ constexpr uint32_t g2_mask(int u) {
    return C == 1 ? (u == 0 ? 0xFFFFFFFFu : (u == 1 ? 0xFCFCFCFCu : (u == 2 ? 0xF0F0F0F0u : 0xC0C0C0C0u)))
         : C == 2 ? (u == 0 ? 0x33333333u : (u == 1 ? 0xCCCCCCCCu : (u == 2 ? 0x30303030u : 0xC0C0C0C0u)))
                  : (0x03030303u << (2 * u));
}
template <int C> __device__ __forceinline__ constexpr int g2_chan(int u) { return C == 1 ? 0 : (C == 2 ? (u & 1) : u); }

// Digit words of four consecutive rows of one channel: rho = base * row[i] (base carries the 2^30), v = round(rho) in
// [-2^30, 2^30].  The addend 1.5 * 2^52 + 0x80808080 rounds to nearest even (as cvt.rni would) and leaves v + 0x80808080 in
// the low word; its bytes ^ 0x80 ARE the four signed base-256 digits of v (adding 128 to every digit makes them unsigned
// bytes without carries between them; ^ 0x80 takes the 128 off again in two's complement).  A 4 x 4 byte transpose (8 PRMT)
// then puts digit d of the four rows into the word of column d (0..3 Re, 4..7 Im).  FULL: all four rows exist; else rows
// i >= nv get zero digits.
template <bool FULL>
__device__ __forceinline__ void g2_item_digits(const double2 base, const double2 (&row)[4], uint32_t nv, uint32_t (&w)[8]) {
    constexpr double kRound = 6755399441055744.0 + 2155905152.0;
    uint32_t vr[4], vi[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const double re = base.x * row[i].x - base.y * row[i].y, im = base.x * row[i].y + base.y * row[i].x;
        vr[i] = (uint32_t)__double2loint(re + kRound) ^ 0x80808080u;
        vi[i] = (uint32_t)__double2loint(im + kRound) ^ 0x80808080u;
        if (!FULL && (uint32_t)i >= nv) { vr[i] = 0u; vi[i] = 0u; }
    }
    const uint32_t r01l = __byte_perm(vr[0], vr[1], 0x5140), r23l = __byte_perm(vr[2], vr[3], 0x5140);
    const uint32_t r01h = __byte_perm(vr[0], vr[1], 0x7362), r23h = __byte_perm(vr[2], vr[3], 0x7362);
    const uint32_t i01l = __byte_perm(vi[0], vi[1], 0x5140), i23l = __byte_perm(vi[2], vi[3], 0x5140);
    const uint32_t i01h = __byte_perm(vi[0], vi[1], 0x7362), i23h = __byte_perm(vi[2], vi[3], 0x7362);
    w[0] = __byte_perm(r01l, r23l, 0x5410); w[1] = __byte_perm(r01l, r23l, 0x7632);
    w[2] = __byte_perm(r01h, r23h, 0x5410); w[3] = __byte_perm(r01h, r23h, 0x7632);
    w[4] = __byte_perm(i01l, i23l, 0x5410); w[5] = __byte_perm(i01l, i23l, 0x7632);
    w[6] = __byte_perm(i01h, i23h, 0x5410); w[7] = __byte_perm(i01h, i23h, 0x7632);
}

// CPW = chunks per consumer warp (1, 2 or 4: rows of <= 8, 16, 32 chunks); a tile has KG = 4 / CPW groups of 32 rows
template <int C, bool SIGN_MAG, int CPW, int NCLS>
__global__ void __launch_bounds__(kG2Threads, NCLS == 1 ? 2 : 1) gen2_kernel(     // (two CTAs per SM: <= 80 registers; several classes: one CTA, <= 168)
const __grid_constant__ Gen2Params P) {
    static_assert(NCLS == 1 || C == 4, "several byte classes per launch: words of 8 / 16 channels");
    if (!P.input_ready) pdl_wait();
    using Cfg = G2Cfg<C, CPW, NCLS>;
    constexpr int KG = Cfg::KG, RT = Cfg::RT, CT = Cfg::CT;
    constexpr int DEPTH = Cfg::TILES, DIGD = Cfg::DIGITS;
    constexpr int NG = Cfg::NG, NT = Cfg::THREADS;                            // generator warps, threads of the CTA
    constexpr uint32_t DIG_BYTES = Cfg::DIG_BYTES;
    extern __shared__ __align__(128) unsigned char g2_smem[];
    unsigned char* ring = g2_smem;                                            // [DEPTH] padded sample tiles
    unsigned char* dig = ring + (size_t)DEPTH * kG2StageBytes;                // [DIGD][CT] digit matrices (Cfg::DIG_CH words each)
    double2* tab_s = reinterpret_cast<double2*>(dig + (size_t)DIGD * DIG_BYTES);    // [C][4 tiles][4][RT / 4] row phasors of a batch (TAB_SMEM)
    uint64_t* bars = reinterpret_cast<uint64_t*>(dig + (size_t)DIGD * DIG_BYTES + (Cfg::TAB_SMEM ? Cfg::TAB_BYTES : 0u));   // full, empty [DEPTH]; digfull, digempty [DIGD]; ticket
    uint32_t* dig_tile = reinterpret_cast<uint32_t*>(bars + 2 * DEPTH + 2 * DIGD + 1);   // [DIGD] tile of a digit entry
    uint32_t* s_gen = dig_tile + DIGD;                                         // [0] sequence number, [1] dft_started seen, [3] arrival, [4], [5] first claims, [6], [7] next batch (second generator warp)
    __shared__ long long s_rsum[kG2MaxCh][2];                                  // sum of the quantised phasors of this CTA's valid rows
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t full0 = smem_u32(bars), empty0 = full0 + 8 * DEPTH, dfull0 = empty0 + 8 * DEPTH,
                   dempty0 = dfull0 + 8 * DIGD, seqbar = dempty0 + 8 * DIGD;

    if (tid == 0) {
        for (int s = 0; s < DEPTH; ++s) {
            mbar_init(full0 + 8 * s, 33);                 // 32 cp.async arrivals of the loader + 1 plain arrival (it has seen the digits)
            mbar_init(empty0 + 8 * s, kG2Consumers);
        }
        for (int e = 0; e < DIGD; ++e) { mbar_init(dfull0 + 8 * e, 1); mbar_init(dempty0 + 8 * e, kG2Consumers); }
        mbar_init(seqbar, 1);
#pragma unroll
        for (int c = 0; c < (int)kG2MaxCh; ++c) { s_rsum[c][0] = 0; s_rsum[c][1] = 0; }
    }
    __syncthreads();

    int acc[NCLS][CPW][4][4];         // [byte class][chunk of this warp][combination u][C fragment]
#pragma unroll
    for (int q = 0; q < NCLS; ++q)
#pragma unroll
        for (int c = 0; c < CPW; ++c)
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int k = 0; k < 4; ++k) acc[q][c][u][k] = 0;

    if (warp >= 1 && warp <= NG) {
        const int gw = warp - 1;                                  // generator warp gw: tiles gw, gw + NG, ... of the CTA's sequence
        // ---------------- generators: own the CTA's tile sequence; digit matrices of a batch of tiles ----------------
        // Batches: the CTA's own index and index + grid first (no round trip before the first tiles), then claims from the
        // launch's counter, each issued two batches ahead.  A claimed batch is always processed: claiming stops with the first
        // batch number past the end.
        // The four digit bytes of a column for rows 4q .. 4q+3 are one 32-bit word of the B fragment (row group q / 8, K slots
        // 4 (q % 8) ..; columns 0..3 = Re digits, 4..7 = Im digits).
        // Work items: (channel, four consecutive rows), g2_item_digits.  A tile has Q = RT / 4 row quads per channel.  A lane
        // serves ONE channel (one batch phasor, one set of digit sums): with CT Q <= 32 items lane l takes quad l % Q of
        // channel l / Q; else 32 / CT lanes share a channel and take its quads in turn (KI items per lane and tile).
        constexpr int Q = RT / 4, KI = Cfg::KI;
        constexpr int LC = Cfg::LC, DIG_CH = Cfg::DIG_CH, TAB_CH = Cfg::TAB_CH;   // lanes per channel; padded per-channel strides
        const int g_ch = lane / LC, g_sub = lane % LC;                          // channel, first quad (quads g_sub + k LC)
        const bool g_on = g_ch < CT;
        const int g_chc = g_on ? g_ch : 0;
        // the row phasors of a batch, from shared memory (an L2 round trip per tile is what these warps cannot afford): row
        // r = RT j + 4 q + i of channel c at [c][j][i][q], so that the lanes of a load are neighbours
        if (Cfg::TAB_SMEM) {
            for (int x = lane + 32 * gw; x < CT * 4 * RT; x += 32 * NG) {                       // (each warp a third of the entries)
                const int c = x / (4 * RT), r = x % (4 * RT);
                tab_s[c * TAB_CH + ((r / RT) * 4 + (r & 3)) * Q + (r % RT) / 4] = __ldg(P.gtab + (size_t)c * kG2TabStride + r);
            }
            asm volatile("bar.sync 1, %0;" ::"n"(32 * NG) : "memory");
        }
        auto cmul = [](const double2 a, const double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); };
        // column sums of the digit matrices of this lane's items: the sum of the quantised phasors over the CTA's rows, which
        // the level offset -3 of every sample needs (rows that do not exist have zero digits; four digits of at most 128 per item: no overflow)
        int dsum[8];
#pragma unroll
        for (int d = 0; d < 8; ++d) dsum[d] = 0;
        // The CTA's batch sequence: positions 0 .. n_static-1 are its own (index + position * grid: most of the launch,
        // no round trips), the rest are claims from the launch's counter.  Claims are two positions ahead -- the first two
        // were made by the ticket thread -- so a claim has two batches' time to come back.
        uint32_t it = 0, pos = 0;
        uint32_t batch = blockIdx.x;
        uint32_t pend[2] = {kG2Invalid, kG2Invalid};           // lane 0: claims in flight for positions pos + 1, pos + 2 (by parity)
        bool have_seq = false;
        uint32_t* ctr = nullptr;
        const uint32_t dyn0 = P.n_static * gridDim.x;          // first claimed batch number
        const double2* g_tab = P.gtab + (size_t)g_chc * kG2TabStride;
        auto load_tabs = [&](uint32_t b, double2& thi, double2& tlo) {
            thi = __ldg(g_tab + kG2TabRows + kG2TabLo + ((b >> 8) & (kG2TabHi - 1u)));
            tlo = __ldg(g_tab + kG2TabRows + (b & 255u));
        };
        double2 thi, tlo;
        load_tabs(batch, thi, tlo);
        while (batch < P.n_batches) {
            const uint32_t tile0 = batch * kG2Batch;
            const uint32_t nt = P.n_tiles - tile0 < kG2Batch ? P.n_tiles - tile0 : kG2Batch;
            const bool all_rows = (uint64_t)(tile0 + kG2Batch) * RT <= P.n_rows;      // (all but the last batch of a piece)
            double2 base = cmul(cmul(P.base0[g_chc], thi), tlo);                      // batch phasor of this lane's channel, scaled by 2^30
            base.x *= 1073741824.0; base.y *= 1073741824.0;
            // the next batch of the sequence, and its table entries on their way while this batch is built
            uint32_t nbatch;
            if (pos + 1 < P.n_static) {
                nbatch = blockIdx.x + (pos + 1) * gridDim.x;
            } else if (gw != 0) {
                nbatch = 0;           // (from warp 1, below)
            } else {
                if (!have_seq) {      // (the ticket and its two claims have long arrived by now)
                    mbar_wait(seqbar, 0u);
                    ctr = P.ctr + 2 * (s_gen[0] % kTailSlots);
                    pend[0] = s_gen[4 + ((pos + 1) & 1u)]; pend[1] = s_gen[4 + ((pos + 2) & 1u)];
                    if (pos + 1 != P.n_static) pend[1] = kG2Invalid;          // (n_static == 0 never happens: host)
                    have_seq = true;
                }
                nbatch = __shfl_sync(0xFFFFFFFFu, pend[0], 0);
                // a claimed batch is always processed: claiming stops with the first batch number past the end
                pend[0] = pend[1]; pend[1] = kG2Invalid;
                if (lane == 0 && nbatch < P.n_batches && pos + 3 - P.n_static < kG2CapBatches) pend[1] = dyn0 + atomicAdd(ctr, 1u);
            }
            if (pos + 1 >= P.n_static) {      // the claimed part of the sequence is warp 1's: one named barrier per batch
                if (gw == 0 && lane == 0) s_gen[6 + (pos & 1u)] = nbatch;
                asm volatile("bar.sync 1, %0;" ::"n"(32 * NG) : "memory");
                nbatch = s_gen[6 + (pos & 1u)];
            }
            load_tabs(nbatch, thi, tlo);
            // digit words of item k of tile jt of the batch
            auto item = [&](uint32_t jt, int k, uint32_t (&w)[8]) {
                const uint32_t quad = (uint32_t)(g_sub + k * LC);
                const uint32_t rb = jt * RT + 4u * quad;                                // first of the item's rows in the batch
                double2 row[4];
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    row[i] = Cfg::TAB_SMEM ? tab_s[g_chc * TAB_CH + (jt * 4 + i) * Q + quad]
                                           : __ldg(g_tab + (rb + i) % kG2TabRows);
                if (all_rows) {
                    g2_item_digits<true>(base, row, 4u, w);
                } else {
                    const uint64_t r_abs = (uint64_t)tile0 * RT + rb;
                    const uint32_t nv = r_abs < P.n_rows ? (P.n_rows - r_abs < 4u ? (uint32_t)(P.n_rows - r_abs) : 4u) : 0u;   // valid rows from there on
                    g2_item_digits<false>(base, row, nv, w);
                }
            };
            auto store = [&](uint32_t* dg, int k, const uint32_t (&w)[8]) {
                const uint32_t quad = (uint32_t)(g_sub + k * LC);
                // word of (channel, row group, column, K slots 4 q7 ..), q7 = quad % 8: at column * 8 + 2 (q7 % 4) + q7 / 4, so that the
                // two B-fragment registers of consumer lane (g = column, t = q7 % 4) are ONE 64-bit load at word 2 * lane; row groups
                // are kG2DigRG = 72 words apart, which spreads the 32 quads of a single-channel tile over all banks
                uint32_t* d = dg + g_ch * DIG_CH + (quad >> 3) * kG2DigRG + 2u * (quad & 3u) + ((quad >> 2) & 1u);
#pragma unroll
                for (int col = 0; col < 8; ++col) {
                    d[col * 8] = w[col];
                    dsum[col] = __dp4a((int)w[col], 0x01010101, dsum[col]);
                }
            };
            constexpr uint32_t JS = (uint32_t)NG;               // tile step of this warp inside a batch
            const uint32_t jf = ((uint32_t)gw + NG - it % NG) % NG;               // its first tile: tiles of the CTA's sequence in turn
            if constexpr (KI == 1) {
                // two tiles at a time: their (independent) phasor chains overlap; computed before the entry is waited for
#pragma unroll 1
                for (uint32_t j0 = jf; j0 < nt; j0 += 2 * JS) {
                    uint32_t w[2][8];
#pragma unroll
                    for (uint32_t ju = 0; ju < 2; ++ju)
                        item(j0 + ju * JS < kG2Batch ? j0 + ju * JS : kG2Batch - 1u, 0, w[ju]);      // (past the batch: computed, not stored)
#pragma unroll
                    for (uint32_t ju = 0; ju < 2; ++ju) {
                        const uint32_t j = j0 + ju * JS;
                        if (j < nt) {
                            const uint32_t e = (it + j) % DIGD, ph = ((it + j) / DIGD) & 1u;
                            mbar_wait(dempty0 + 8 * e, ph ^ 1u);          // the consumers are done with the entry's previous tile
                            if (g_on) store(reinterpret_cast<uint32_t*>(dig + (size_t)e * DIG_BYTES), 0, w[ju]);
                            if (lane == 0) dig_tile[e] = tile0 + j;
                            __syncwarp();
                            if (lane == 0) mbar_arrive(dfull0 + 8 * e);
                        }
                    }
                }
            } else {
                // several items per lane and tile: item by item into the entry (two in flight)
#pragma unroll 1
                for (uint32_t j = jf; j < nt; j += JS) {
                    const uint32_t e = (it + j) % DIGD, ph = ((it + j) / DIGD) & 1u;
                    mbar_wait(dempty0 + 8 * e, ph ^ 1u);
                    uint32_t* dg = reinterpret_cast<uint32_t*>(dig + (size_t)e * DIG_BYTES);
#pragma unroll 1
                    for (int k = 0; k < KI; k += 2) {
                        uint32_t w[2][8];
                        item(j, k, w[0]);
                        item(j, k + 1, w[1]);
                        if (g_on) { store(dg, k, w[0]); store(dg, k + 1, w[1]); }
                    }
                    if (lane == 0) dig_tile[e] = tile0 + j;
                    __syncwarp();
                    if (lane == 0) mbar_arrive(dfull0 + 8 * e);
                }
            }
            it += nt;
            batch = nbatch; ++pos;
        }
        {   // terminator: the entry after the last tile carries "no tile"
            const uint32_t e = it % DIGD, ph = (it / DIGD) & 1u;
            mbar_wait(dempty0 + 8 * e, ph ^ 1u);
            if (lane == 0 && gw == 0) { dig_tile[e] = kG2Invalid; mbar_arrive(dfull0 + 8 * e); }
        }
        {
            long long re = (long long)dsum[0] + ((long long)dsum[1] << 8) + ((long long)dsum[2] << 16) + ((long long)dsum[3] << 24);
            long long im = (long long)dsum[4] + ((long long)dsum[5] << 8) + ((long long)dsum[6] << 16) + ((long long)dsum[7] << 24);
#pragma unroll
            for (int sh = LC / 2; sh > 0; sh >>= 1) {          // the lanes of a channel: LC consecutive ones
                re += __shfl_xor_sync(0xFFFFFFFFu, re, sh);
                im += __shfl_xor_sync(0xFFFFFFFFu, im, sh);
            }
            if (g_sub == 0 && g_on) {         // (every generator warp holds a part)
                atomicAdd(reinterpret_cast<unsigned long long*>(&s_rsum[g_ch][0]), (unsigned long long)re);
                atomicAdd(reinterpret_cast<unsigned long long*>(&s_rsum[g_ch][1]), (unsigned long long)im);
            }
        }
    } else if (warp == 0) {
        // ---------------- loader: copy each tile as it lies, 512 contiguous bytes per instruction ----------------
        // The ticket is taken: the next launch may become resident (its CTAs take the slots this launch leaves free or frees).
        mbar_wait(seqbar, 0u);
        pdl_release();
        // this lane's 16 bytes of warp load 0: row and column in the padded tile
        const uint32_t q0 = ((uint32_t)lane * 16u) / P.row_bytes, col0 = ((uint32_t)lane * 16u) % P.row_bytes;
        const bool pow2 = P.chunks == 8u * CPW && P.row_stride == P.row_bytes;  // 8, 16 or 32 chunks, rows contiguous: 512 bytes = whole rows
        for (uint32_t it = 0;; ++it) {
            const uint32_t e = it % DIGD, phe = (it / DIGD) & 1u;
            const uint32_t s = it % DEPTH, ph = (it / DEPTH) & 1u;
            mbar_wait(dfull0 + 8 * e, phe);
            const uint32_t tile = dig_tile[e];
            mbar_wait(empty0 + 8 * s, ph ^ 1u);
            if (tile == kG2Invalid) {
                cp_async_arrive_noinc(full0 + 8 * s);
                if (lane == 0) mbar_arrive(full0 + 8 * s);
                break;
            }
            const uint64_t row0 = (uint64_t)tile * RT;
            const uint32_t rows = P.n_rows - row0 < (uint64_t)RT ? (uint32_t)(P.n_rows - row0) : (uint32_t)RT;
            const uint32_t stage = smem_u32(ring) + s * kG2StageBytes;
            const unsigned char* src = P.data + row0 * P.row_stride + P.col_off + (uint32_t)lane * 16u;
            if (rows == (uint32_t)RT && pow2) {
                // row_bytes = 128 CPW: a warp load covers 4 / CPW rows
                g2_copy_tile<0, 32, (4u / CPW) * (128u * CPW + 16u)>(stage + q0 * (128u * CPW + 16u) + col0, src);
            } else {
                uint32_t q = q0, col = col0;
                const uint32_t valid_bytes = rows * P.row_bytes;
                const unsigned char* rows_src = P.data + row0 * P.row_stride + P.col_off;
                for (uint32_t o = (uint32_t)lane * 16u; o < valid_bytes; o += 512u) {
                    cp_async16(stage + q * P.pitch + col, rows_src + (uint64_t)q * P.row_stride + col);
                    col += 512u;
                    while (col >= P.row_bytes) { col -= P.row_bytes; ++q; }
                }
            }
            cp_async_arrive_noinc(full0 + 8 * s);
            if (lane == 0) mbar_arrive(full0 + 8 * s);              // (release: what this warp has seen -- the digits -- is visible to whoever sees "full")
        }
    } else {
        // ---------------- consumers: warp cw owns chunks CPW cw .. CPW cw + CPW - 1 of every row ----------------
        const int cw = warp - 1 - NG;
        if (cw == 0 && lane == 0) {
            // ticket: sequence number of this launch, derived on the device (pcal_tail.cuh, "Pipelining"); taken before the
            // loader lets the dependent grid start.  The slot's previous user (launch seq - kTailSlots) must have finished
            // before the slot's counters are touched.
            const unsigned long long tk = atomicAdd(&P.st->tick, 1ull);   // (ticket and acquire load in flight together: pcal_tail.cuh)
            uint32_t done, x;
            ld_acquire_done_started(P.st, done, x);
            const uint32_t sq = (uint32_t)(tk / gridDim.x);
            s_gen[0] = sq; s_gen[1] = x;
            if ((int32_t)(done - (sq - kTailSlots + 1u)) < 0)
                while ((int32_t)(ld_acquire_u32(&P.st->n_done) - (sq - kTailSlots + 1u)) < 0) __nanosleep(64);
            // the generator's first two claims (positions n_static, n_static + 1 of its sequence; slot by position parity)
            uint32_t* ctr = P.ctr + 2 * (sq % kTailSlots);
            const uint32_t d0 = P.n_static * gridDim.x + atomicAdd(ctr, 1u), d1 = P.n_static * gridDim.x + atomicAdd(ctr, 1u);
            s_gen[4 + (P.n_static & 1u)] = d0; s_gen[4 + ((P.n_static + 1u) & 1u)] = d1;
            mbar_arrive(seqbar);
        }
        __syncwarp();
        const uint32_t first = (uint32_t)(cw * CPW);
        const uint32_t my = smem_u32(ring) + (uint32_t)lane * P.pitch + first * 16u;
        const uint32_t nch = P.chunks > first ? (P.chunks - first < (uint32_t)CPW ? P.chunks - first : (uint32_t)CPW) : 0u;   // this warp's chunks
        const uint32_t kg_step = 32u * P.pitch;
        // one chunk of one row group: byte column -> four masked operands -> four MMAs
        // (several classes: the masked operand meets the digits of channel u of EVERY class -- an MMA's 16 byte columns hold all
        //  classes, each lane keeps the sums of its own; the B fragments come straight from the digit entry, `dgk` = row group kg)
        auto chunk_mma = [&](int c, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, const uint32_t (&bf)[C][2], const uint32_t* dgk) {
            if (SIGN_MAG) {
                a0 = signmag_to_offset_binary(a0); a1 = signmag_to_offset_binary(a1);
                a2 = signmag_to_offset_binary(a2); a3 = signmag_to_offset_binary(a3);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t m = g2_mask<C>(u);
                const int ch = g2_chan<C>(u);
                if constexpr (NCLS == 1) {
                    if (m == 0xFFFFFFFFu) mma_u8s8_k32(acc[0][c][u], a0, a1, a2, a3, bf[ch][0], bf[ch][1]);
                    else mma_u8s8_k32(acc[0][c][u], a0 & m, a1 & m, a2 & m, a3 & m, bf[ch][0], bf[ch][1]);
                } else {
                    const uint32_t x0 = a0 & m, x1 = a1 & m, x2 = a2 & m, x3 = a3 & m;
#pragma unroll
                    for (int q = 0; q < NCLS; ++q) {
                        const uint2 b = *reinterpret_cast<const uint2*>(dgk + (q * C + ch) * Cfg::DIG_CH + 2 * lane);
                        mma_u8s8_k32(acc[q][c][u], x0, x1, x2, x3, b.x, b.y);
                    }
                }
            }
        };
        for (uint32_t it = 0;; ++it) {
            const uint32_t e = it % DIGD;
            const uint32_t s = it % DEPTH, ph = (it / DEPTH) & 1u;
            mbar_wait(full0 + 8 * s, ph);
            const uint32_t tile = dig_tile[e];
            const uint32_t* dg32 = reinterpret_cast<const uint32_t*>(dig + (size_t)e * DIG_BYTES);
            auto load_bf = [&](int kg, uint32_t (&bf)[C][2]) {
                if constexpr (NCLS == 1) {
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        const uint2 b = *reinterpret_cast<const uint2*>(dg32 + c * Cfg::DIG_CH + kg * kG2DigRG + 2 * lane);
                        bf[c][0] = b.x; bf[c][1] = b.y;
                    }
                }
            };
            const uint32_t base = my + s * kG2StageBytes;
            if (nch == (uint32_t)CPW) {
                // complete rows (the usual case): every operand load of the tile is issued before the first MMA
                uint32_t a[KG][CPW][4];
#pragma unroll
                for (int kg = 0; kg < KG; ++kg)
#pragma unroll
                    for (int c = 0; c < CPW; ++c) ldsm_t8_x2(base + kg * kg_step + 16u * c, a[kg][c][0], a[kg][c][1], a[kg][c][2], a[kg][c][3]);
                if (tile == kG2Invalid) break;
                if constexpr (NCLS == 1) {
#pragma unroll
                    for (int kg = 0; kg < KG; ++kg) {
                        uint32_t bf[C][2];
                        load_bf(kg, bf);
#pragma unroll
                        for (int c = 0; c < CPW; ++c) chunk_mma(c, a[kg][c][0], a[kg][c][1], a[kg][c][2], a[kg][c][3], bf, dg32 + kg * kG2DigRG);
                    }
                } else {
                    // several classes: per row group and combination u the B fragments of channel u of every class are loaded
                    // once (2 NCLS registers) and meet the masked operands of all of this warp's chunks
#pragma unroll
                    for (int kg = 0; kg < KG; ++kg) {
                        if (SIGN_MAG) {
#pragma unroll
                            for (int c = 0; c < CPW; ++c)
#pragma unroll
                                for (int r = 0; r < 4; ++r) a[kg][c][r] = signmag_to_offset_binary(a[kg][c][r]);
                        }
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            uint32_t bq[NCLS][2];
#pragma unroll
                            for (int q = 0; q < NCLS; ++q) {
                                const uint2 b = *reinterpret_cast<const uint2*>(dg32 + kg * kG2DigRG + (q * C + g2_chan<C>(u)) * Cfg::DIG_CH + 2 * lane);
                                bq[q][0] = b.x; bq[q][1] = b.y;
                            }
                            const uint32_t m = g2_mask<C>(u);
#pragma unroll
                            for (int c = 0; c < CPW; ++c) {
                                const uint32_t x0 = a[kg][c][0] & m, x1 = a[kg][c][1] & m, x2 = a[kg][c][2] & m, x3 = a[kg][c][3] & m;
#pragma unroll
                                for (int q = 0; q < NCLS; ++q) mma_u8s8_k32(acc[q][c][u], x0, x1, x2, x3, bq[q][0], bq[q][1]);
                            }
                        }
                    }
                }
            } else {
                if (tile == kG2Invalid) break;
#pragma unroll
                for (int kg = 0; kg < KG; ++kg) {
                    uint32_t bf[C][2];
                    load_bf(kg, bf);
#pragma unroll
                    for (int c = 0; c < CPW; ++c) {
                        if ((uint32_t)c < nch) {
                            uint32_t a0, a1, a2, a3;
                            ldsm_t8_x2(base + kg * kg_step + 16u * c, a0, a1, a2, a3);
                            chunk_mma(c, a0, a1, a2, a3, bf, dg32 + kg * kG2DigRG);
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) { mbar_arrive(empty0 + 8 * s); mbar_arrive(dempty0 + 8 * e); }
        }
    }
    __syncthreads();                  // every role is done: the ring becomes the per-position result array
    const uint32_t seq = s_gen[0], slot = seq % kTailSlots;
    uint32_t* ctr = P.ctr + 2 * slot;

    // ---- epilogue: digit sums -> exact per-position int64 (re, im) * 2^30 -> red.add into the launch's accumulators ----
    long long* pos_s = reinterpret_cast<long long*>(ring);                  // [kG2Fields][2]
    if (warp >= 1 + NG) {
        const int cw = warp - 1 - NG, g = lane >> 2, t = lane & 3;
#pragma unroll
        for (int c = 0; c < CPW; ++c) {
            // this lane's byte columns (g, g + 8 of every chunk) belong to one byte class: the sums of that class
            const uint32_t kcls = (uint32_t)g % P.cls_count - P.cls;          // class index inside the launch (wraps when below it)
            const bool mine = kcls < (uint32_t)NCLS;                           // (8 / 16 channels: the bytes of this launch's channels)
            int A[4][4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    A[u][k] = acc[0][c][u][k];
#pragma unroll
                    for (int q = 1; q < NCLS; ++q) if (kcls == (uint32_t)q) A[u][k] = acc[q][c][u][k];
                }
            // field sums from the combination sums (exact: every U is a sum of non-negative multiples of the S)
            int S[4][4];              // [field f][C fragment], field f scaled by 4^f
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (C == 1) {
                    S[0][k] = A[0][k] - A[1][k]; S[1][k] = A[1][k] - A[2][k];
                    S[2][k] = A[2][k] - A[3][k]; S[3][k] = A[3][k];
                } else if (C == 2) {
                    S[0][k] = A[0][k] - A[2][k]; S[1][k] = A[1][k] - A[3][k];
                    S[2][k] = A[2][k]; S[3][k] = A[3][k];
                } else {
                    S[0][k] = A[0][k]; S[1][k] = A[1][k]; S[2][k] = A[2][k]; S[3][k] = A[3][k];
                }
            }
#pragma unroll
            for (int f = 0; f < 4; ++f)
#pragma unroll
                for (int hi = 0; hi < 2; ++hi) {
                    // C fragment: [2 hi], [2 hi + 1] = digit columns 2t, 2t+1 of M row g + 8 hi.  Columns 0..3 = Re digits,
                    // 4..7 = Im digits: lane t = 0 (2) holds the low half of Re (Im), lane t = 1 (3) the high half.
                    const int c0 = S[f][2 * hi] >> (2 * f), c1 = S[f][2 * hi + 1] >> (2 * f);
                    const int x0 = __shfl_down_sync(0xFFFFFFFFu, c0, 1), x1 = __shfl_down_sync(0xFFFFFFFFu, c1, 1);
                    const long long v = (long long)c0 + ((long long)c1 << 8) + ((long long)x0 << 16) + ((long long)x1 << 24);
                    const int ri = t >> 1;                                    // 0: Re, 1: Im (lanes t = 0 and t = 2 own the results)
                    if (!(t & 1)) {
                        const uint32_t bytecol = (uint32_t)(cw * CPW + c) * 16u + (uint32_t)g + 8u * hi;
                        const uint32_t F = 4u * bytecol + (uint32_t)f;
                        pos_s[2 * F + ri] = mine ? 2 * v - 3 * s_rsum[kcls * C + f % C][ri] : 0;    // codes 0..3 -> levels 2 code - 3
                    }
                }
        }
    }
    __syncthreads();
    const uint32_t nval = 2u * 64u * P.chunks;                              // values of the positions that exist
    {
        long long* dst = P.posacc + (size_t)slot * 2 * kG2Fields;
        for (uint32_t i = tid; i < nval; i += NT) { const long long v = pos_s[i]; if (v) red_add_s64(dst + i, v); }
    }
    __syncthreads();                  // every thread's reds happen before thread 0's release below
    if (tid == 0) s_gen[3] = arrive_acq_rel(ctr + 1);
    __syncthreads();
    if (s_gen[3] != gridDim.x - 1u) return;

    // ---- final stage (the CTA that arrived last): positions -> bins, ragged tail, accumulate into the context ----
    // (first the loads whose latency the rest can hide: the progress counters, the accumulators, the position factors)
    uint32_t seen_done = 0, seen_dft = 0;
    if (tid == 0) { seen_done = ld_acquire_u32(&P.st->n_done); seen_dft = ld_acquire_u32(&P.st->dft_finished); }
    long long* gacc = P.posacc + (size_t)slot * 2 * kG2Fields;
    for (uint32_t i = tid; i < nval; i += NT) { pos_s[i] = __ldcg(gacc + i); gacc[i] = 0; }     // and ready for the slot's next launch
    const uint32_t pairs = (uint32_t)CT * P.n_bins, n_tail = (uint32_t)(P.n_total - P.n_body);
    double2* sP = reinterpret_cast<double2*>(ring + 2 * kG2Fields * sizeof(long long));               // [pairs] (fused DFT)
    const uint32_t dft_x = s_gen[1];
    __syncthreads();
    bool waited = false;
    auto wait_for_P = [&]() {
        if (tid == 0) {
            uint32_t a = seen_done, b = seen_dft;
            while (a != seq || (int32_t)(b - dft_x) < 0) {
                __nanosleep(32);
                a = ld_acquire_u32(&P.st->n_done); b = ld_acquire_u32(&P.st->dft_finished);
            }
        }
        __syncthreads();
    };
    const FastDiv dBins(P.n_bins);                            // (dividends below 2^24: pcal_common.cuh)
    const uint32_t tau_first = dBins.mod(2u * P.n_bins - P.n0_mod_bins - dBins.mod(P.tau0));      // time offset of bin 0 in this launch's columns
    for (uint32_t pp0 = 0; pp0 < pairs; pp0 += NT) {          // uniform trip count
        const uint32_t pp = pp0 + tid;
        const bool mine = pp < pairs;
        uint32_t c = 0u, b = 0u;
        if (mine) dBins.divmod(pp, c, b);
        double re = 0.0, im = 0.0;
        if (mine) {
            const double2* tw = P.tw + (size_t)c * P.span_t + P.tau0;
            const uint32_t n_tau = 64u * P.chunks / ((uint32_t)C * P.cls_count);       // time offsets in this launch's columns
            // tau0 + tau = b - n0 (mod N_bins), in order
            uint32_t tau = b + tau_first; if (tau >= P.n_bins) tau -= P.n_bins;
            for (; tau < n_tau; tau += P.n_bins) {
                const uint32_t F = (tau * P.cls_count + P.cls + c / C) * C + c % C;       // (class of channel c: c / C)
                const double xr = (double)pos_s[2 * F] * (1.0 / 1073741824.0), xi = (double)pos_s[2 * F + 1] * (1.0 / 1073741824.0);
                const double2 w = __ldg(tw + tau);
                re += xr * w.x - xi * w.y;
                im += xr * w.y + xi * w.x;
            }
            if (n_tail && P.do_tail) {     // samples n_body .. n_total-1 (less than one row), exactly reduced phases
                const uint32_t bb0 = (uint32_t)((P.n0 + P.n_body) % P.n_bins);
                for (uint32_t tt = (b + P.n_bins - bb0) % P.n_bins; tt < n_tail; tt += P.n_bins) {
                    const double v = decode_tail(KIND_2BIT, SIGN_MAG ? 1 : 0, P.tail, tt, P.c_base + c, P.c_real);
                    const double2 ph = phasor_neg(mulmod_u64(P.Foff[c], P.n0 + P.n_body + tt, P.Fs), P.Fs);
                    re += v * ph.x; im += v * ph.y;
                }
            }
        }
        if (!waited) { wait_for_P(); waited = true; }
        if (!mine) continue;
        const uint32_t po = P.c_base * P.n_bins + pp;             // (c_base + c, b) in the context's arrays
        if (!P.overwrite) { const double2 cur = __ldcg(P.P + po); re += cur.x; im += cur.y; }
        P.P[po] = make_double2(re, im);
        if (P.fuse_dft) sP[pp] = make_double2(re, im);
        if (P.P_copy) P.P_copy[po] = make_double2(re, im);
    }
    if (P.fuse_dft) {   // T[c] = DFT(P[c]), channel by channel, from shared memory
        __syncthreads();
        double2* sY = sP + pairs;
        dft_in_cta(sP, sY, P.W, (uint32_t)CT, P.n_bins, P.dft_n1, P.k_shift % P.n_bins, P.T_dev, P.T_host, NT);
    }
    if (tid == 0) { ctr[0] = 0u; ctr[1] = 0u; }
    __syncthreads();
    if (tid == 0) st_release_u32(&P.st->n_done, seq + 1u);             // P is final for this launch; the slot is free
}

}  // namespace pcal
