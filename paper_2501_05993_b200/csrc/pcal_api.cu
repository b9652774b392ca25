// pcal_api.cu -- host side of libpcal: the C ABI declared in include/pcal.h.
// Validates, derives the geometry (N_bins, rotator lengths, fold period), builds tables in long
// double on the host, and enqueues the kernels of pcal_fold.cuh / pcal_gen.cuh / pcal_post.cuh on
// the caller's stream.  No CPU compute path: every step of the hot path runs in those kernels.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "../../include/pcal_noalloc.h"
#include "pcal_ctx.h"
#include "pcal_fold.cuh"
#include "pcal_gen.cuh"
#include "pcal_post.cuh"
#include "pcal_gen_mma.cuh"
#include "pcal_gen2.cuh"
#include "pcal_analysis.cuh"
#include "pcal_genstudy.cuh"

using namespace pcal;
typedef unsigned __int128 u128;

namespace {

constexpr uint64_t kMaxFoldPeriod = 1ull << 22;   // LUT mode: M*C accumulators at most
constexpr uint32_t kMaxSlotGroups = 2048;         // LUT mode: q at most
constexpr uint64_t kMaxLutEntries = 1ull << 22;
constexpr uint32_t kMaxBins = 4096;
constexpr uint32_t kMaxIterPerLaunch = 2048;      // keeps the 16-bit lanes of fold_2bit exact
constexpr size_t kStageBytes = 128ull << 20;
constexpr uint64_t kMaxTailEntries = 1ull << 17;  // fused tail: q * C * N_bins per-group bins at most (2 MiB)
constexpr uint32_t kTailMaxReplicas = 32;         // fused tail: the fold period is doubled until R <= this

uint64_t gcd64(uint64_t a, uint64_t b) { while (b) { uint64_t t = a % b; a = b; b = t; } return a; }
// lcm with saturation
uint64_t lcm_sat(uint64_t a, uint64_t b, uint64_t cap) {
    if (a == 0 || b == 0) return 0;
    u128 l = (u128)(a / gcd64(a, b)) * b;
    return l > cap ? cap + 1 : (uint64_t)l;
}
uint64_t to_uhz(double f_hz) { return (uint64_t)llround(f_hz * 1e6); }
uint64_t mulmod_host(uint64_t a, uint64_t b, uint64_t m) { return (uint64_t)(((u128)a * b) % m); }
double2 phasor_neg_host(uint64_t k, uint64_t m) {
    const long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)m;
    return make_double2((double)cosl(ang), (double)(-sinl(ang)));
}

}  // namespace

static void free_tables(pcal_ctx* c) {
    cudaFree(c->d_lut); cudaFree(c->d_lut_off); cudaFree(c->d_lut_len);
    cudaFree(c->d_partial); cudaFree(c->d_gen_partial);
    cudaFree(c->d_val); cudaFree(c->d_cnt); cudaFree(c->d_G); cudaFree(c->d_tail_state);
    cudaFree(c->d_g2_rtab); cudaFree(c->d_g2_tw); cudaFree(c->d_g2_ctr); cudaFree(c->d_g2_posacc);
    c->d_g2_rtab = c->d_g2_tw = nullptr; c->d_g2_ctr = nullptr; c->d_g2_posacc = nullptr;
    c->d_cnt = nullptr; c->d_G = nullptr; c->d_tail_state = nullptr;
    c->d_lut = nullptr; c->d_lut_off = c->d_lut_len = nullptr;
    c->d_partial = nullptr; c->d_gen_partial = nullptr;
    c->d_val = nullptr;
}

extern "C" const char* pcal_strerror(int code) {
    switch (code) {
        case PCAL_OK: return "ok";
        case PCAL_ERR_INVALID: return "invalid argument";
        case PCAL_ERR_ALIGNMENT: return "pointer or segment length not aligned";
        case PCAL_ERR_STATE: return "call not legal in this state";
        case PCAL_ERR_UNSUPPORTED: return "unsupported configuration";
        case PCAL_ERR_DEVICE: return "CUDA device error";
        case PCAL_ERR_NOMEM: return "out of memory";
        case PCAL_ERR_LIMIT: return "size exceeds the fixed scratch of the no-allocation entry point (N_bins <= 1024, one channel)";
        default: return "unknown error";
    }
}

extern "C" int pcal_create(pcal_ctx** out, double f_s_hz, double f_comb_hz, double f_offset_hz,
                           int bits, int encoding, int n_channels) {
    if (!out) return PCAL_ERR_INVALID;
    *out = nullptr;
    if (!(f_s_hz > 0) || !(f_comb_hz > 0) || !(f_offset_hz >= 0) || !(f_offset_hz < f_s_hz)) return PCAL_ERR_INVALID;
    const uint64_t Fs = to_uhz(f_s_hz), Fc = to_uhz(f_comb_hz), Fo = to_uhz(f_offset_hz);
    if (Fs == 0 || Fc == 0 || Fs % Fc != 0 || Fs / Fc < 2 || Fs >= (1ull << 62)) return PCAL_ERR_INVALID;
    if (Fs / Fc > kMaxBins) return PCAL_ERR_UNSUPPORTED;
    int kind;
    if (bits == 2 && (encoding == PCAL_ENC_OFFSET_BINARY || encoding == PCAL_ENC_SIGN_MAG)) kind = KIND_2BIT;
    else if (bits == 8 && encoding == PCAL_ENC_TWOS_COMPLEMENT) kind = KIND_I8;
    else if (bits == 32 && encoding == PCAL_ENC_IEEE_FLOAT) kind = KIND_F32;
    else return PCAL_ERR_INVALID;
    if (n_channels < 1 || n_channels > PCAL_MAX_CHANNELS || (n_channels & (n_channels - 1))) return PCAL_ERR_INVALID;
    if (n_channels > 1 && bits != 2) return PCAL_ERR_INVALID;

    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PCAL_ERR_DEVICE; }
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); return PCAL_ERR_DEVICE; }

    pcal_ctx* c = new (std::nothrow) pcal_ctx();
    if (!c) return PCAL_ERR_NOMEM;
    memset(c, 0, sizeof(*c));
    c->Fs = Fs; c->Fcomb = Fc;
    for (int i = 0; i < n_channels; ++i) c->Foff[i] = Fo;
    c->bits = bits; c->enc = encoding; c->C = n_channels; c->kind = kind;
    c->sign_mag = (encoding == PCAL_ENC_SIGN_MAG);
    c->n_bins = (uint32_t)(Fs / Fc);
    c->rot_req = PCAL_ROT_AUTO;
    c->device = dev; c->sm_count = sms;
    const size_t nb = (size_t)c->n_bins * n_channels;
    bool ok = cudaMalloc(&c->d_P, nb * sizeof(double2)) == cudaSuccess &&
              cudaMalloc(&c->d_T, nb * sizeof(double2)) == cudaSuccess &&
              cudaMalloc(&c->d_tmp, nb * sizeof(double2)) == cudaSuccess &&
              cudaMalloc(&c->d_Pint, nb * sizeof(long long)) == cudaSuccess &&
              cudaMalloc(&c->d_W, (size_t)c->n_bins * sizeof(double2)) == cudaSuccess &&
              cudaMallocHost(&c->h_pinned, nb * sizeof(double2)) == cudaSuccess &&
              cudaMalloc(&c->d_summary, (size_t)n_channels * kNSummary * sizeof(double)) == cudaSuccess &&
              cudaMalloc(&c->d_B, nb * sizeof(double2)) == cudaSuccess &&
              cudaMallocHost(&c->h_ana, (size_t)n_channels * kNSummary * sizeof(double) + nb * sizeof(double2)) == cudaSuccess;
    if (ok) {
        std::vector<double2> W(c->n_bins);
        for (uint32_t k = 0; k < c->n_bins; ++k) W[k] = phasor_neg_host(k, c->n_bins);
        // (synchronous copy from pageable memory: complete on return.  The accumulators are zeroed lazily, on the
        //  stream of the first call that needs them: zero_pending.)
        ok = cudaMemcpy(c->d_W, W.data(), W.size() * sizeof(double2), cudaMemcpyHostToDevice) == cudaSuccess;
        c->zero_pending = true;
    }
    if (ok && 2 * (size_t)c->n_bins * sizeof(double2) > 48 * 1024)
        ok = cudaFuncSetAttribute(dft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)(2 * (size_t)c->n_bins * sizeof(double2))) == cudaSuccess;
    if (!ok) { cudaGetLastError(); pcal_destroy(c); return PCAL_ERR_DEVICE; }
    *out = c;
    return PCAL_OK;
}

extern "C" void pcal_destroy(pcal_ctx* c) {
    if (!c) return;
    free_tables(c);
    cudaFree(c->d_P); cudaFree(c->d_T); cudaFree(c->d_tmp); cudaFree(c->d_Pint); cudaFree(c->d_W);
    cudaFree(c->d_stage);
    cudaFreeHost(c->h_pinned); cudaFreeHost(c->h_ana);
    cudaFree(c->d_summary); cudaFree(c->d_B);
    if (c->ev) { for (cudaEvent_t e : *c->ev) cudaEventDestroy(e); delete c->ev; }
    cudaGetLastError();
    delete c;
}

extern "C" int pcal_set_channel_offsets(pcal_ctx* c, const double* f) {
    if (!c || !f) return PCAL_ERR_INVALID;
    if (c->started) return PCAL_ERR_STATE;
    uint64_t tmp[PCAL_MAX_CHANNELS];
    for (int i = 0; i < c->C; ++i) {
        if (!(f[i] >= 0)) return PCAL_ERR_INVALID;
        tmp[i] = to_uhz(f[i]);
        if (tmp[i] >= c->Fs) return PCAL_ERR_INVALID;
    }
    memcpy(c->Foff, tmp, sizeof(uint64_t) * c->C);
    c->prepared = false;
    return PCAL_OK;
}

extern "C" int pcal_set_rotator(pcal_ctx* c, int mode) {
    if (!c || mode < PCAL_ROT_AUTO || mode > PCAL_ROT_GENERATOR) return PCAL_ERR_INVALID;
    if (c->started) return PCAL_ERR_STATE;
    c->rot_req = mode; c->prepared = false;
    return PCAL_OK;
}

extern "C" int pcal_set_k_shift(pcal_ctx* c, int k) {
    if (!c || k < 0 || (uint32_t)k >= c->n_bins) return PCAL_ERR_INVALID;
    if (c->started) return PCAL_ERR_STATE;
    c->k_shift = k; c->prepared = false;
    return PCAL_OK;
}

extern "C" int pcal_set_input_ready(pcal_ctx* c, int ready) {
    if (!c) return PCAL_ERR_INVALID;
    c->input_ready = ready != 0;
    return PCAL_OK;
}

extern "C" int pcal_set_start_index(pcal_ctx* c, uint64_t n_start) {
    if (!c) return PCAL_ERR_INVALID;
    if (c->started) return PCAL_ERR_STATE;
    c->n_processed = n_start;
    return PCAL_OK;
}

extern "C" int pcal_info(const pcal_ctx* c, pcal_info_t* info) {
    if (!c || !info) return PCAL_ERR_INVALID;
    memset(info, 0, sizeof(*info));
    info->n_channels = c->C; info->n_bins = (int32_t)c->n_bins; info->bits = c->bits; info->encoding = c->enc;
    info->rotator_requested = c->rot_req; info->rotator_in_effect = c->prepared ? c->rot_eff : 0;
    info->integer_exact = (c->prepared && c->all_zero && c->kind != KIND_F32) ? 1 : 0;
    info->k_shift = c->k_shift;
    info->n_processed = c->n_processed;
    info->fold_period = c->prepared && c->rot_eff == PCAL_ROT_LUT ? c->M : 0;
    for (int i = 0; i < c->C; ++i) {
        const uint64_t Fe = (c->Foff[i] + (uint64_t)c->k_shift * c->Fcomb) % c->Fs;
        const uint64_t nrot = Fe ? c->Fs / gcd64(c->Fs, Fe) : 1;
        info->lut_len[i] = lcm_sat(c->n_bins, nrot, ~0ull >> 1);
    }
    info->kernel_launches = c->launches;
    return PCAL_OK;
}

// fold_2bit_kernel instantiations: <SIGN_MAG, loads per block, CTAs per SM>.  The default was
// chosen on the B200 (profiles/); PCAL_FOLD2_VARIANT=u4b3|u4b4|u8b2 overrides it for tuning runs.
typedef void (*fold2_fn)(const FoldParams);
static fold2_fn pick_fold2(bool sm) {
    const char* v = getenv("PCAL_FOLD2_VARIANT");
    if (v && !strcmp(v, "u4b4")) return sm ? fold_2bit_kernel<true, 4, 4> : fold_2bit_kernel<false, 4, 4>;
    if (v && !strcmp(v, "u8b2")) return sm ? fold_2bit_kernel<true, 8, 2> : fold_2bit_kernel<false, 8, 2>;
    if (v && !strcmp(v, "u8b3")) return sm ? fold_2bit_kernel<true, 8, 3> : fold_2bit_kernel<false, 8, 3>;
    return sm ? fold_2bit_kernel<true, 4, 3> : fold_2bit_kernel<false, 4, 3>;
}

// ---------------------------------------------------------------------------------------------
// Lazy set-up: decide LUT vs generator, derive the geometry, build the rotator tables.
// ---------------------------------------------------------------------------------------------
static uint32_t dft_ctas(const pcal_ctx* c);
// N = N1 * N2 for the two-stage DFT of the fused tails: N1 = the largest divisor of N not above sqrt(N)
static uint32_t dft_n1_of(uint32_t n) {
    uint32_t best = 1;
    for (uint32_t d = 1; d * d <= n; ++d) if (n % d == 0) best = d;
    return best;
}

// the gen2_kernel instantiation of a context: <channels per byte, SIGN_MAG, chunks per consumer warp, byte classes per launch>
typedef void (*gen2_kfn)(const Gen2Params);
template <int C, int CPW, int NCLS>
static gen2_kfn gen2_pick_sm(bool sm) { return sm ? gen2_kernel<C, true, CPW, NCLS> : gen2_kernel<C, false, CPW, NCLS>; }
template <int C>
static gen2_kfn gen2_pick_cpw(uint32_t cpw, bool sm) {
    return cpw == 1 ? gen2_pick_sm<C, 1, 1>(sm) : (cpw == 2 ? gen2_pick_sm<C, 2, 1>(sm) : gen2_pick_sm<C, 4, 1>(sm));
}
// words of 8 / 16 channels: a time sample is 2 / 4 bytes ("classes" of four channels).  A launch serves g2_ncls classes: all of
// them where the accumulators fit (rows of <= 16 chunks), else one class per launch and as many passes over the data.
static int gen2_ck(const pcal_ctx* c) { return c->C < 4 ? c->C : 4 * (int)c->g2_ncls; }       // channels per launch
static gen2_kfn gen2_kernel_of(const pcal_ctx* c) {
    const bool sm = c->sign_mag != 0;
    if (c->C == 1) return gen2_pick_cpw<1>(c->g2_cpw, sm);
    if (c->C == 2) return gen2_pick_cpw<2>(c->g2_cpw, sm);
    if (c->g2_ncls == 2) return c->g2_cpw == 1 ? gen2_pick_sm<4, 1, 2>(sm) : gen2_pick_sm<4, 2, 2>(sm);
    if (c->g2_ncls == 4) return c->g2_cpw == 1 ? gen2_pick_sm<4, 1, 4>(sm) : gen2_pick_sm<4, 2, 4>(sm);
    return gen2_pick_cpw<4>(c->g2_cpw, sm);
}
template <int C>
static size_t gen2_smem_c(uint32_t cpw) { return cpw == 1 ? gen2_smem_bytes<C, 1, 1>() : (cpw == 2 ? gen2_smem_bytes<C, 2, 1>() : gen2_smem_bytes<C, 4, 1>()); }
static size_t gen2_smem_of(const pcal_ctx* c) {
    if (c->g2_ncls == 2) return c->g2_cpw == 1 ? gen2_smem_bytes<4, 1, 2>() : gen2_smem_bytes<4, 2, 2>();
    if (c->g2_ncls == 4) return c->g2_cpw == 1 ? gen2_smem_bytes<4, 1, 4>() : gen2_smem_bytes<4, 2, 4>();
    return c->C == 1 ? gen2_smem_c<1>(c->g2_cpw) : (c->C == 2 ? gen2_smem_c<2>(c->g2_cpw) : gen2_smem_c<4>(c->g2_cpw));
}
static const void* gen2_fn(const pcal_ctx* c) { return reinterpret_cast<const void*>(gen2_kernel_of(c)); }

static int prepare(pcal_ctx* c) {
    if (c->prepared) return PCAL_OK;
    free_tables(c);
    c->all_zero = true;
    uint64_t total_lut = 0;
    for (int i = 0; i < c->C; ++i) {
        c->Feff[i] = (c->Foff[i] + (uint64_t)c->k_shift * c->Fcomb) % c->Fs;
        c->nrot[i] = c->Feff[i] ? c->Fs / gcd64(c->Fs, c->Feff[i]) : 1;   // eq. 2.4
        if (c->Feff[i]) c->all_zero = false;
        total_lut += c->nrot[i] > kMaxLutEntries ? kMaxLutEntries + 1 : c->nrot[i];
    }
    c->spv = c->kind == KIND_F32 ? 4u : (c->kind == KIND_I8 ? 16u : 64u / (uint32_t)c->C);
    c->F = c->kind == KIND_F32 ? 4u : (c->kind == KIND_I8 ? 16u : 64u);
    c->gen_spt = c->kind == KIND_F32 ? 4u : 16u;

    uint64_t M = lcm_sat(c->n_bins, c->spv, kMaxFoldPeriod);
    for (int i = 0; i < c->C; ++i) M = M > kMaxFoldPeriod ? M : lcm_sat(M, c->nrot[i], kMaxFoldPeriod);
    bool lut_ok = M <= kMaxFoldPeriod && total_lut <= kMaxLutEntries;
    uint32_t q = 0;
    if (lut_ok) {
        const uint64_t S = M / c->spv;
        const uint64_t qq = S / gcd64(S, 32);
        lut_ok = qq <= kMaxSlotGroups;
        q = (uint32_t)qq;
    }
    const char* gm = getenv("PCAL_GEN_MMA");       // =0: FFMA2 kernel of pcal_gen.cuh for every sample type (A/B runs, tests)
    c->gen_mma = c->C == 1 && c->kind == KIND_I8 && kMmaSpan % c->n_bins == 0 && !(gm && gm[0] == '0');
    // 2-bit samples: pcal_gen2.cuh.  A row is a multiple of lcm(N_bins, time samples per 16 bytes) time samples.
    // PCAL_GEN2=0 or PCAL_GEN_MMA=0 selects the FFMA2 kernel instead (single channel; A/B runs, tests).
    c->gen2 = false;
    {
        const char* g2 = getenv("PCAL_GEN2");
        if (c->kind == KIND_2BIT && !(g2 && g2[0] == '0') && !(gm && gm[0] == '0')) {
            const uint64_t lam = lcm_sat(c->n_bins, 64u / (uint32_t)c->C, 1u << 20);      // <= 4096 * 64 time samples
            {
                // the shortest row with at least 8 chunks (one per consumer warp): few positions, few accumulators.  A row of
                // more than 32 chunks (2048 fields) is served in column blocks of 32 chunks, one launch each.
                const uint32_t lam_chunks = (uint32_t)(lam * (uint64_t)c->C / 64u);
                // Several channels: as many rows of <= 16 chunks as fit (the generator warp's work per tile is per channel and row).
                const char* mc = getenv("PCAL_G2_CHUNKS");       // (tests: other row lengths)
                uint32_t m = lam_chunks >= 8u ? 1u : (8u + lam_chunks - 1u) / lam_chunks;
                if (c->C > 1 && 16u / lam_chunks > m) m = 16u / lam_chunks;
                if (mc && (uint32_t)atoi(mc) / lam_chunks >= 1u) m = (uint32_t)atoi(mc) / lam_chunks;
                c->gen2 = true;
                c->g2_span_t = (uint32_t)lam * m;
                c->g2_chunks = lam_chunks * m;
                c->g2_blocks = (c->g2_chunks + 31u) / 32u;
                c->g2_cpw = c->g2_chunks <= 8u ? 1u : (c->g2_chunks <= 16u ? 2u : 4u);
                c->g2_rt = 32u * (4u / c->g2_cpw);
                // byte classes per launch (8 / 16 channels): all of them when a thread's accumulators fit (PCAL_G2_NCLS: A/B runs, tests)
                c->g2_ncls = 1;
                if (c->C > 4 && c->g2_cpw <= 2u && c->g2_blocks == 1u) c->g2_ncls = (uint32_t)c->C / 4u;
                if (const char* nc = getenv("PCAL_G2_NCLS")) { const uint32_t v = (uint32_t)atoi(nc); if (c->g2_ncls > 1 && (v == 1 || v == 2) && v <= c->g2_ncls) c->g2_ncls = v; }
            }
        }
    }
    // FFMA2 kernel (float32; int8 when N_bins does not divide 2048): a CTA iteration covers the largest multiple of
    // lcm(N_bins, samples per load) that its 256 threads hold
    {
        const uint64_t unit = lcm_sat(c->n_bins, c->gen_spt, 1u << 20), cap = (uint64_t)kThreads * c->gen_spt;
        c->gen_span = unit <= cap ? (uint32_t)(unit * (cap / unit)) : 0u;
    }
    const bool gen_ok = c->gen2 || (c->C == 1 && (c->gen_mma || c->gen_span != 0));
    int mode;
    if (c->all_zero) mode = PCAL_ROT_LUT;
    else if (c->rot_req == PCAL_ROT_LUT) mode = lut_ok ? PCAL_ROT_LUT : 0;
    else if (c->rot_req == PCAL_ROT_GENERATOR) mode = gen_ok ? PCAL_ROT_GENERATOR : 0;
    else mode = lut_ok ? PCAL_ROT_LUT : (gen_ok ? PCAL_ROT_GENERATOR : 0);
    if (!mode) return PCAL_ERR_UNSUPPORTED;
    c->rot_eff = mode;

    if (mode == PCAL_ROT_LUT) {
        int occ = 0;
        size_t elem = 0;
        if (c->kind == KIND_2BIT) { c->fold2 = pick_fold2(c->sign_mag != 0); occ = occupancy_of(c->fold2, 0); elem = 2; }
        else if (c->kind == KIND_I8) { occ = occupancy_of(fold_i8_kernel, 0); elem = 4; }
        else { occ = occupancy_of(fold_f32_kernel, 0); elem = 8; }
        if (occ < 1) return PCAL_ERR_DEVICE;
        const uint32_t slots = (uint32_t)(c->sm_count * occ);
        // Fused tail (pcal_tail.cuh): one CTA sums the R replicas of a slot group, so R is kept small by
        // folding modulo a larger multiple of L (any multiple is a valid period): more, smaller groups.
        const uint64_t pairs = (uint64_t)c->n_bins * c->C;
        const char* nf = getenv("PCAL_NO_FUSED_TAIL");
        c->fused = !(nf && nf[0] == '1') && (uint64_t)q * pairs <= kMaxTailEntries;
        while (c->fused && slots / q > kTailMaxReplicas) {
            const uint64_t M2 = M * 2, S2 = M2 / c->spv, q2 = S2 / gcd64(S2, 32);
            if (M2 > kMaxFoldPeriod || q2 > kMaxSlotGroups || q2 * pairs > kMaxTailEntries) break;
            M = M2; q = (uint32_t)q2;
        }
        c->q = q; c->M = M;
        c->R = slots / q ? slots / q : 1;
        if (c->fused) {
            // leave room for the CTAs of the two previous launches that are still in their tail (q+1 each)
            // and for the CTAs of a DFT kernel: the next launch must become resident in one wave
            const uint32_t reserve = 2 * (q + 1) + dft_ctas(c) + 8;
            if (slots > reserve + q) c->R = (slots - reserve) / q;
            // Half of that when it still gives every SM a CTA: the CTAs of TWO consecutive launches then fit on the machine, so a
            // launch streams while its predecessor is in its prologue or tail instead of waiting for the predecessor's slots
            // (measured, steps back to back: config 1 4.5 (or 6.0: two regimes) -> 3.6 us, config 2 11.3 -> 10.0 us, config 3
            // 19.5 -> 18.4 us, config 4 40.4 -> 36.0 us; a launch on its own is 5-20 % slower).  PCAL_FOLD_FULL_GRID=1: the full grid.
            const char* fg = getenv("PCAL_FOLD_FULL_GRID");
            if (!(fg && fg[0] == '1') && slots > reserve + 2 * q && (slots - reserve) / (2 * q) * q >= (uint32_t)c->sm_count)
                c->R = (slots - reserve) / (2 * q);
            const uint32_t W = 32u * c->spv, per = W / c->n_bins ? W / c->n_bins : 1u;
            uint32_t tpp = 1; while (tpp * 2 <= per && tpp < 32) tpp *= 2;
            c->tail_tpp = tpp;
            const size_t ns = kTailSlots;
            CU(cudaMalloc(&c->d_cnt, ns * ((size_t)c->q + 2) * sizeof(uint32_t)));
            CU(cudaMemsetAsync(c->d_cnt, 0, ns * ((size_t)c->q + 2) * sizeof(uint32_t), c->stream));
            CU(cudaMalloc(&c->d_G, ns * (size_t)c->q * pairs * sizeof(double2)));
            CU(cudaMalloc(&c->d_tail_state, sizeof(TailState)));
            CU(cudaMemsetAsync(c->d_tail_state, 0, sizeof(TailState), c->stream));
        }
        c->grid = c->q * c->R;
        c->partial_slot_bytes = (size_t)c->grid * c->F * 32 * elem;
        CU(cudaMalloc(&c->d_partial, c->partial_slot_bytes * (c->fused ? kTailSlots : 1)));
        CU(cudaMalloc(&c->d_val, (size_t)c->q * c->F * 32 * sizeof(double)));
        // rotate_fold_kernel: a warp per (channel, bin) pair, or the whole CTA when a pair has many elements
        const uint64_t per_pair = (uint64_t)c->q * 32u * c->spv / c->n_bins;
        c->rot_tpp = per_pair > 256 ? (uint32_t)kPostThreads : 32u;
        // rotator tables (eq. 2.4), one per channel, built in long double
        std::vector<double2> lut;
        std::vector<uint32_t> off(c->C), len(c->C);
        for (int i = 0; i < c->C; ++i) {
            off[i] = (uint32_t)lut.size(); len[i] = (uint32_t)c->nrot[i]; c->lut_off_h[i] = off[i];
            for (uint64_t r = 0; r < c->nrot[i]; ++r) lut.push_back(phasor_neg_host(mulmod_host(r, c->Feff[i], c->Fs), c->Fs));
            c->lut_len[i] = c->nrot[i];
        }
        CU(cudaMalloc(&c->d_lut, lut.size() * sizeof(double2)));
        CU(cudaMalloc(&c->d_lut_off, c->C * sizeof(uint32_t)));
        CU(cudaMalloc(&c->d_lut_len, c->C * sizeof(uint32_t)));
        CU(cudaMemcpyAsync(c->d_lut, lut.data(), lut.size() * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(c->d_lut_off, off.data(), c->C * sizeof(uint32_t), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(c->d_lut_len, len.data(), c->C * sizeof(uint32_t), cudaMemcpyHostToDevice, c->stream));
    } else {
        int occ = 0;
        if (c->gen2) {
            // tables in long double from exactly reduced phases: stride phasors per row, position factors per time offset
            const uint32_t C = (uint32_t)c->C, span = c->g2_span_t;
            std::vector<double2> rtab((size_t)C * kG2TabStride), tw((size_t)C * span);
            const uint64_t D = (uint64_t)kG2Batch * c->g2_rt * span;       // samples per batch
            for (uint32_t ch = 0; ch < C; ++ch) {
                double2* g = rtab.data() + (size_t)ch * kG2TabStride;
                for (uint32_t r = 0; r < kG2TabRows; ++r) g[r] = phasor_neg_host(mulmod_host((uint64_t)r * span, c->Feff[ch], c->Fs), c->Fs);
                for (uint32_t k = 0; k < kG2TabLo; ++k) g[kG2TabRows + k] = phasor_neg_host(mulmod_host(D * k % c->Fs, c->Feff[ch], c->Fs), c->Fs);
                for (uint32_t k = 0; k < kG2TabHi; ++k) g[kG2TabRows + kG2TabLo + k] = phasor_neg_host(mulmod_host(D * 256 * k % c->Fs, c->Feff[ch], c->Fs), c->Fs);
                for (uint32_t t = 0; t < span; ++t) tw[(size_t)ch * span + t] = phasor_neg_host(mulmod_host(t, c->Feff[ch], c->Fs), c->Fs);
            }
            CU(cudaMalloc(&c->d_g2_rtab, rtab.size() * sizeof(double2)));
            CU(cudaMalloc(&c->d_g2_tw, tw.size() * sizeof(double2)));
            CU(cudaMalloc(&c->d_g2_ctr, kTailSlots * 2 * sizeof(uint32_t)));
            CU(cudaMalloc(&c->d_g2_posacc, (size_t)kTailSlots * 2 * kG2Fields * sizeof(long long)));
            CU(cudaMalloc(&c->d_tail_state, sizeof(TailState)));
            CU(cudaMemcpyAsync(c->d_g2_rtab, rtab.data(), rtab.size() * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
            CU(cudaMemcpyAsync(c->d_g2_tw, tw.data(), tw.size() * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
            CU(cudaMemsetAsync(c->d_g2_ctr, 0, kTailSlots * 2 * sizeof(uint32_t), c->stream));
            CU(cudaMemsetAsync(c->d_g2_posacc, 0, (size_t)kTailSlots * 2 * kG2Fields * sizeof(long long), c->stream));
            CU(cudaMemsetAsync(c->d_tail_state, 0, sizeof(TailState), c->stream));
            c->gen_smem = gen2_smem_of(c);
            const void* fn = gen2_fn(c);
            CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->gen_smem));
            CU(cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
            c->gen_grid = (uint32_t)c->sm_count;           // half-SM CTAs, one per SM: consecutive launches share the SMs
            c->prepared = true;
            return PCAL_OK;
        }
        if (c->gen_mma) { c->gen_smem = gen_mma_smem_bytes<KIND_I8>(); CU(cudaFuncSetAttribute(gen_mma_kernel<KIND_I8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->gen_smem)); occ = occupancy_of(gen_mma_kernel<KIND_I8, false>, c->gen_smem); }
        else if (c->kind == KIND_2BIT) { c->gen_smem = gen_smem_bytes<KIND_2BIT>(); CU(cudaFuncSetAttribute(gen_kernel<KIND_2BIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->gen_smem)); occ = occupancy_of(gen_kernel<KIND_2BIT>, c->gen_smem); }
        else if (c->kind == KIND_I8) { c->gen_smem = gen_smem_bytes<KIND_I8>(); CU(cudaFuncSetAttribute(gen_kernel<KIND_I8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->gen_smem)); occ = occupancy_of(gen_kernel<KIND_I8>, c->gen_smem); }
        else { c->gen_smem = gen_smem_bytes<KIND_F32>(); CU(cudaFuncSetAttribute(gen_kernel<KIND_F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->gen_smem)); occ = occupancy_of(gen_kernel<KIND_F32>, c->gen_smem); }
        if (occ < 1) return PCAL_ERR_DEVICE;
        c->gen_grid = (uint32_t)(c->sm_count * occ);
        // float32: one CTA per SM and launch (64 KB of loads in flight each): the CTAs of consecutive launches share the SMs, so the
        // prologue and the tail of one launch hide under the streaming of the next (64 MB per step: 17 -> 12 us; 1 GB: 154 -> 150 us)
        if (!c->gen_mma && c->kind == KIND_F32) c->gen_grid = (uint32_t)c->sm_count;
        // ... and one CTA per TWO SMs when the first segment (or period) the context sees is short (< 128 MB, ~20 us of streaming):
        // the fixed cost of a CTA (ticket, tables, epilogue: ~4 us) is then spread over twice the data, and four launches are
        // resident together instead of two (the paper's shape, 64 MB per step: 11.3 -> 9.7 us; on its own 27 -> 31 us).  The grid
        // stays as chosen for the life of the geometry: the launch sequence numbers are tickets / grid (pcal_tail.cuh).
        if (!c->gen_mma && c->kind == KIND_F32 && c->first_bytes && c->first_bytes < (128ull << 20) && c->sm_count >= 2)
            c->gen_grid = (uint32_t)c->sm_count / 2u;
        if (const char* gg = getenv("PCAL_GEN_GRID")) { if (!c->gen_mma && atoi(gg) > 0) c->gen_grid = (uint32_t)atoi(gg); }   // tuning runs only
        // The fused tail pays while the partial bins of a launch are few (its finishing CTAs hold the slots of CTAs of the next
        // launch, whose tile assignment is static); config 5 (296 CTAs x 1024 bins) keeps the separate post and DFT kernels.
        c->gen_fused = !c->gen_mma && (uint64_t)c->gen_grid * c->n_bins <= (1u << 16);       // (FFMA2 kernel only)
        CU(cudaMalloc(&c->d_gen_partial, (size_t)(c->gen_fused ? kTailSlots : 1) * c->gen_grid * c->n_bins * sizeof(double2)));
        CU(cudaMalloc(&c->d_g2_ctr, kTailSlots * 2 * sizeof(uint32_t)));     // arrival counters of the generator tail
        CU(cudaMalloc(&c->d_tail_state, sizeof(TailState)));
        CU(cudaMemsetAsync(c->d_g2_ctr, 0, kTailSlots * 2 * sizeof(uint32_t), c->stream));
        CU(cudaMemsetAsync(c->d_tail_state, 0, sizeof(TailState), c->stream));
    }
    c->prepared = true;
    return PCAL_OK;
}

// Accumulators hold zeros after pcal_reset only lazily: the first post kernel of the next
// pcal_extract overwrites them; any other reader zeroes them first.
static int ensure_zeroed(pcal_ctx* c) {
    if (!c->zero_pending) return PCAL_OK;
    const uint32_t n = c->n_bins * (uint32_t)c->C;
    zero_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(c->d_P, c->d_Pint, n);
    c->launches += 1;
    CU(cudaGetLastError());
    c->zero_pending = false;
    return PCAL_OK;
}

static uint32_t log2_u32(uint32_t v) { uint32_t l = 0; while ((1u << l) < v) ++l; return l; }

// one launch group of the LUT / zero-offset path over n time samples starting at data
static int extract_piece_lut(pcal_ctx* c, const uint8_t* data, uint64_t n, cudaStream_t st) {
    const uint64_t n_bytes = n * (uint64_t)c->bits * c->C / 8;
    const uint64_t n_vec = n_bytes / 16;
    if (n_vec) {
        FoldParams fp;
        fp.data = reinterpret_cast<const uint4*>(data); fp.n_vec = n_vec; fp.q = c->q; fp.R = c->R;
        const uint64_t NC = (n_vec + 31) / 32, NSR = (NC + c->q - 1) / c->q;
        uint64_t it = (NSR + (uint64_t)c->R * kWarps - 1) / ((uint64_t)c->R * kWarps);
        it = (it + kFoldGroup - 1) / kFoldGroup * kFoldGroup;
        fp.n_iter = (uint32_t)it;
        fp.partial = c->d_partial;            // fused tail: slot 0 of the ring; the kernel picks its slot
        const uint64_t grid_threads = (uint64_t)c->R * kWarps * c->q * 32u;
        fp.n_quot = (uint32_t)(n_vec / grid_threads); fp.n_rem = n_vec % grid_threads;
        fp.input_ready = c->input_ready ? 1 : 0;
        TailParams& tp = fp.tail;
        memset(&tp, 0, sizeof(tp));
        if (c->fused) {
            tp.enabled = 1;
            tp.cnt = c->d_cnt; tp.G = c->d_G; tp.st = c->d_tail_state; tp.partial_stride = c->partial_slot_bytes;
            if (c->fuse_req) {
                tp.fuse_dft = 1; tp.dft_n1 = dft_n1_of(c->n_bins); tp.k_shift = (uint32_t)c->k_shift; tp.W = c->d_W;
                tp.T_dev = c->fuse_T_dev ? c->fuse_T_dev : c->d_T; tp.T_host = c->fuse_out; tp.P_copy = c->fuse_P_copy;
            }
            tp.lut = c->d_lut;
            for (int i = 0; i < c->C; ++i) { tp.lut_off[i] = c->lut_off_h[i]; tp.lut_len[i] = (uint32_t)c->nrot[i]; }
            tp.P = c->d_P; tp.Pint = c->d_Pint; tp.tail = data + n_vec * 16;
            tp.n0 = c->n_processed; tp.NT = n_vec * c->spv; tp.n_total = n;
            tp.n0_mod_bins = (uint32_t)(c->n_processed % c->n_bins);
            for (int i = 0; i < c->C; ++i) tp.n0_mod_L[i] = (uint32_t)(c->n_processed % c->nrot[i]);
            tp.cnt_quot = (uint32_t)(n_vec / ((uint64_t)c->q * 32u)); tp.cnt_rem = (uint32_t)(n_vec % ((uint64_t)c->q * 32u));
            tp.C = (uint32_t)c->C; tp.spv = c->spv; tp.spv_log2 = log2_u32(c->spv); tp.n_bins = c->n_bins;
            tp.tpp = c->tail_tpp; tp.kind = c->kind; tp.sign_mag = c->sign_mag;
            tp.integer_exact = (c->all_zero && c->kind != KIND_F32) ? 1 : 0;
            tp.overwrite = c->zero_pending ? 1 : 0;
        }
        prof_mark(c, st);
        if (c->kind == KIND_2BIT) launch_chain(c->fold2, c->grid, kThreads, 0, st, fp);
        else if (c->kind == KIND_I8) launch_chain(fold_i8_kernel, c->grid, kThreads, 0, st, fp);
        else launch_chain(fold_f32_kernel, c->grid, kThreads, 0, st, fp);
        prof_mark(c, st);
        c->launches += 1;
        if (c->fused) {               // the fold kernel's last CTAs did the reduction, the rotation and the tail
            c->zero_pending = false;
            CU(cudaGetLastError());
            return PCAL_OK;
        }
    }
    if (n_vec) {
        ReplicaParams rr;
        rr.partial = c->d_partial; rr.val = c->d_val; rr.q = c->q; rr.R = c->R; rr.F = c->F;
        rr.cnt_quot = (uint32_t)(n_vec / ((uint64_t)c->q * 32u)); rr.cnt_rem = (uint32_t)(n_vec % ((uint64_t)c->q * 32u));
        rr.kind = c->kind;
        const uint32_t total = c->q * c->F * 32u;
        rr.ns = c->R <= 8 ? 1u : (c->R <= 16 ? 2u : (c->R <= 32 ? 4u : 8u));
        const uint32_t epc = (uint32_t)kPostThreads / rr.ns;
        launch_chain(reduce_replicas_kernel, (total + epc - 1) / epc, kPostThreads, 0, st, rr);
        c->launches += 1;
    }
    RotateParams rp;
    rp.val = c->d_val; rp.lut = c->d_lut; rp.lut_off = c->d_lut_off; rp.lut_len = c->d_lut_len;
    rp.P = c->d_P; rp.Pint = c->d_Pint; rp.tail = data + n_vec * 16;
    rp.n0 = c->n_processed; rp.NT = n_vec * c->spv; rp.n_total = n;
    rp.q = c->q; rp.F = c->F; rp.C = (uint32_t)c->C; rp.spv = c->spv; rp.spv_log2 = log2_u32(c->spv);
    rp.n_bins = c->n_bins; rp.tpp = c->rot_tpp; rp.have_val = n_vec ? 1u : 0u;
    rp.kind = c->kind; rp.sign_mag = c->sign_mag;
    rp.integer_exact = (c->all_zero && c->kind != KIND_F32) ? 1 : 0;
    rp.overwrite = c->zero_pending ? 1 : 0;
    rp.release_late = c->fused ? 1 : 0;       // (fused context, piece without a complete vector)
    const uint32_t pairs = c->n_bins * (uint32_t)c->C, ppc = (uint32_t)kPostThreads / c->rot_tpp;
    launch_chain(rotate_fold_kernel, (pairs + ppc - 1) / ppc, kPostThreads, 0, st, rp);
    c->zero_pending = false;
    c->launches += 1;
    CU(cudaGetLastError());
    return PCAL_OK;
}

static int enqueue_dft(pcal_ctx* c, double2* second_dst);
static bool can_fuse_dft(const pcal_ctx* c);

// pcal_gen2.cuh over n time samples starting at data: rows, tail and accumulation in ONE kernel (one launch per group of
// four channels for words of 8 / 16 channels)
static int extract_piece_gen2(pcal_ctx* c, const uint8_t* data, uint64_t n, cudaStream_t st) {
    const int ck = gen2_ck(c);                                     // channels per launch
    const uint32_t n_cls = c->C > 4 ? (uint32_t)c->C / 4u : 1u;    // byte classes of a time sample
    const uint32_t cls_step = c->g2_ncls;                          // classes per launch
    const bool was_pending = c->zero_pending;
    for (uint32_t blk = 0; blk < c->g2_blocks; ++blk)
    for (uint32_t cls = 0; cls < n_cls; cls += cls_step) {
        Gen2Params gp;
        memset(&gp, 0, sizeof(gp));
        const uint64_t n_bytes = n * 2ull * c->C / 8;
        gp.data = data;
        gp.chunks = c->g2_chunks - 32u * blk < 32u ? c->g2_chunks - 32u * blk : 32u;
        gp.row_bytes = gp.chunks * 16u; gp.span_t = c->g2_span_t;
        gp.row_stride = (uint64_t)c->g2_chunks * 16u; gp.col_off = 512ull * blk;
        gp.tau0 = 2048u * blk / (uint32_t)c->C; gp.do_tail = blk == 0 ? 1 : 0;
        gp.pitch = gp.row_bytes + ((gp.chunks & 1u) ? 0u : 16u);      // an odd number of 16-byte chunks
        gp.cls_count = n_cls; gp.cls = cls; gp.c_real = (uint32_t)c->C; gp.c_base = c->C > 4 ? cls * 4u : 0u;
        gp.n_rows = n_bytes / gp.row_stride;
        gp.n_tiles = (uint32_t)((gp.n_rows + c->g2_rt - 1) / c->g2_rt);
        gp.n_batches = (gp.n_tiles + kG2Batch - 1) / kG2Batch;
        gp.n_static = (uint32_t)(3ull * gp.n_batches / (4ull * c->gen_grid));
        if (gp.n_static < 1) gp.n_static = 1;
        gp.Fs = c->Fs;
        for (int i = 0; i < ck; ++i) {
            const int ch = (int)gp.c_base + i;
            gp.Foff[i] = c->Feff[ch];
            gp.base0[i] = phasor_neg_host(mulmod_host(c->n_processed % c->Fs, c->Feff[ch], c->Fs), c->Fs);
        }
        gp.gtab = c->d_g2_rtab + (size_t)gp.c_base * kG2TabStride; gp.tw = c->d_g2_tw + (size_t)gp.c_base * c->g2_span_t;
        gp.ctr = c->d_g2_ctr; gp.posacc = c->d_g2_posacc; gp.st = c->d_tail_state;
        gp.P = c->d_P; gp.tail = data + gp.n_rows * gp.row_stride;
        gp.n0 = c->n_processed; gp.n_body = gp.n_rows * c->g2_span_t; gp.n_total = n;
        gp.n_bins = c->n_bins; gp.n0_mod_bins = (uint32_t)(c->n_processed % c->n_bins);
        gp.overwrite = was_pending && blk == 0 ? 1 : 0; gp.input_ready = c->input_ready ? 1 : 0;
        if (c->fuse_req) {        // (single launch per piece only: can_fuse_dft)
            gp.fuse_dft = 1; gp.dft_n1 = dft_n1_of(c->n_bins); gp.k_shift = (uint32_t)c->k_shift; gp.W = c->d_W;
            gp.T_dev = c->fuse_T_dev ? c->fuse_T_dev : c->d_T; gp.T_host = c->fuse_out; gp.P_copy = c->fuse_P_copy;
        }
        prof_mark(c, st);
        launch_chain(gen2_kernel_of(c), c->gen_grid, kG2Threads, c->gen_smem, st, gp);
        prof_mark(c, st);
        c->launches += 1;
    }
    c->zero_pending = false;
    CU(cudaGetLastError());
    return PCAL_OK;
}

// FFMA2 generator kernel: samples per tile (iterations per tile x samples per iteration)
static uint64_t gen_tile_samples(const pcal_ctx* c) { return (uint64_t)(kTileSamples / (kThreads * c->gen_spt)) * c->gen_span; }

static int extract_piece_gen(pcal_ctx* c, const uint8_t* data, uint64_t n, cudaStream_t st) {
    if (c->gen2) return extract_piece_gen2(c, data, n, st);
    const uint32_t spt = c->gen_spt;
    const uint64_t load_bytes = c->kind == KIND_2BIT ? 4 : 16;
    const uint64_t n_bytes = n * (uint64_t)c->bits / 8;
    uint64_t n_loads = n_bytes / load_bytes;
    if (c->gen_mma) n_loads -= n_loads % (kMmaSpan / spt);        // whole 2048-sample rows; the rest goes to the post kernel
    const uint64_t Fs = c->Fs, Fo = c->Feff[0];
    if (n_loads || c->gen_fused) {   // (fused tail: also for a piece without a complete load -- the kernel's last CTA adds the ragged tail)
        GenParams gp;
        memset(&gp, 0, sizeof(gp));
        gp.data = data; gp.n_loads = n_loads;
        // FFMA2 kernel: a CTA iteration covers gen_span samples (a multiple of N_bins), a tile 2^16 / (kThreads * spt) iterations
        const uint64_t span = c->gen_mma ? (uint64_t)kThreads * spt : c->gen_span;
        const uint64_t tile = c->gen_mma ? kTileSamples : gen_tile_samples(c);
        gp.span = (uint32_t)span;
        gp.n_tiles = (n_loads * spt + tile - 1) / tile;
        gp.n_iters = (n_loads * spt + span - 1) / span;
        gp.Fs = Fs; gp.Foff = Fo;
        gp.k0 = mulmod_host(c->n_processed % Fs, Fo, Fs);
        gp.E = mulmod_host(tile, Fo, Fs);
        gp.D = mulmod_host(c->gen_grid, gp.E, Fs);
        gp.rho = phasor_neg_host(mulmod_host(span, Fo, Fs), Fs);
        gp.rho2 = phasor_neg_host(mulmod_host(2 * span, Fo, Fs), Fs);
        for (uint32_t k = 0; k < 16; ++k) gp.tw[k] = phasor_neg_host(mulmod_host(k, Fo, Fs), Fs);
        gp.n_bins = c->n_bins; gp.sign_mag = c->sign_mag;
        gp.dec_mask = 0x00600000u; gp.dec_one = 0x3F800000u;
        gp.input_ready = c->input_ready ? 1 : 0;
        GenTailParams& tp = gp.tail;
        tp.st = c->gen_fused ? c->d_tail_state : nullptr; tp.cnt = c->d_g2_ctr; tp.partial = c->d_gen_partial; tp.P = c->d_P;
        tp.tail = data + n_loads * load_bytes;
        tp.n0 = c->n_processed; tp.n_body = n_loads * spt; tp.n_total = n; tp.Fs = Fs; tp.Foff = Fo;
        tp.n_bins = c->n_bins; tp.kind = c->kind; tp.sign_mag = c->sign_mag; tp.overwrite = c->zero_pending ? 1 : 0;
        if (c->fuse_req) {
            tp.fuse_dft = 1; tp.dft_n1 = dft_n1_of(c->n_bins); tp.k_shift = (uint32_t)c->k_shift; tp.W = c->d_W;
            tp.T_dev = c->fuse_T_dev ? c->fuse_T_dev : c->d_T; tp.T_host = c->fuse_out; tp.P_copy = c->fuse_P_copy;
        }
        const size_t smem = c->gen_smem;
        prof_mark(c, st);
        if (c->gen_mma) launch_chain(gen_mma_kernel<KIND_I8, false>, c->gen_grid, kThreads, smem, st, gp);
        else if (c->kind == KIND_2BIT) launch_chain(gen_kernel<KIND_2BIT>, c->gen_grid, kThreads, smem, st, gp);
        else if (c->kind == KIND_I8) launch_chain(gen_kernel<KIND_I8>, c->gen_grid, kThreads, smem, st, gp);
        else launch_chain(gen_kernel<KIND_F32>, c->gen_grid, kThreads, smem, st, gp);
        prof_mark(c, st);
        c->launches += 1;
    }
    if (!c->gen_fused) {
        GenPostParams gr;
        gr.partial = c->d_gen_partial; gr.P = c->d_P; gr.tail = data + n_loads * load_bytes;
        gr.n0 = c->n_processed; gr.n_done = n_loads * spt; gr.n_total = n; gr.Fs = Fs; gr.Foff = Fo;
        gr.grid = n_loads ? c->gen_grid : 0; gr.n_bins = c->n_bins; gr.kind = c->kind; gr.sign_mag = c->sign_mag;
        gr.overwrite = c->zero_pending ? 1 : 0;
        launch_chain(post_gen_kernel, (c->n_bins + 31) / 32, kPostThreads, 0, st, gr);
        c->launches += 1;
    }
    c->zero_pending = false;
    CU(cudaGetLastError());
    return PCAL_OK;
}

// PCAL_SMALL_PIECES=1 (tests only): see extract_segment.  Read per call (tests toggle it), but cheaply.
static bool small_pieces() {
    const char* sp = getenv("PCAL_SMALL_PIECES");
    return sp && sp[0] == '1';
}

// time samples per launch: bounded per-thread trip count (LUT path) / bounded resync table or claims per CTA (generator path).
// PCAL_SMALL_PIECES=1 (tests only) shrinks the limits so that a few million samples already span several
// launches; the arithmetic is unchanged.
static uint64_t piece_samples(const pcal_ctx* c, bool small) {
    if (c->rot_eff == PCAL_ROT_LUT) return (uint64_t)(small ? 16u : kMaxIterPerLaunch) * c->R * kWarps * c->q * 32ull * c->spv;
    if (c->gen2) return (uint64_t)(small ? 2 : kG2CapBatches * kG2Batch / 2) * c->gen_grid * c->g2_rt * c->g2_span_t;   // <= half of what the CTAs may claim
    return (uint64_t)(small ? 2 : kGenMaxTiles) * c->gen_grid * (c->gen_mma ? (uint64_t)kTileSamples : gen_tile_samples(c));   // resync table: <= 256 tiles per CTA
}

static int extract_segment(pcal_ctx* c, const uint8_t* p, uint64_t n_samples) {
    const uint64_t piece = piece_samples(c, small_pieces());
    uint64_t done = 0;
    while (done < n_samples) {
        const uint64_t n = n_samples - done < piece ? n_samples - done : piece;
        const uint8_t* base = p + done * (uint64_t)c->bits * c->C / 8;
        const int r = c->rot_eff == PCAL_ROT_LUT ? extract_piece_lut(c, base, n, c->stream)
                                                 : extract_piece_gen(c, base, n, c->stream);
        if (r != PCAL_OK) return r;
        c->n_processed += n;
        done += n;
    }
    return PCAL_OK;
}

extern "C" int pcal_extract(pcal_ctx* c, const void* dev_samples, uint64_t n_samples, void* cuda_stream) {
    if (!c) return PCAL_ERR_INVALID;
    if (n_samples == 0) return PCAL_OK;
    if (!dev_samples) return PCAL_ERR_INVALID;
    if ((uintptr_t)dev_samples & 15u) return PCAL_ERR_ALIGNMENT;
    if ((n_samples * (uint64_t)c->bits * c->C) % 8) return PCAL_ERR_ALIGNMENT;
    c->stream = (cudaStream_t)cuda_stream;       // prepare() issues its set-up copies on the caller's stream
    if (!c->prepared) c->first_bytes = n_samples * (uint64_t)c->bits * c->C / 8;
    const int rc = prepare(c);
    if (rc != PCAL_OK) return rc;
    c->started = true;
    return extract_segment(c, reinterpret_cast<const uint8_t*>(dev_samples), n_samples);
}

// A time series of integrations (112 pulses of 10 s each): period k covers the
// samples [k, k+1) * n_per_period of the segment; the accumulators restart at every period while the
// sample index -- hence the rotator phase -- runs on.
extern "C" int pcal_extract_series(pcal_ctx* c, const void* dev_samples, uint64_t n_per_period, uint32_t n_periods,
                                   void* cuda_stream, double* dev_out_tones, double* dev_out_folded) {
    if (!c || !dev_out_tones) return PCAL_ERR_INVALID;
    if (n_periods == 0 || n_per_period == 0) return PCAL_OK;
    if (!dev_samples) return PCAL_ERR_INVALID;
    const uint64_t bits_per_period = n_per_period * (uint64_t)c->bits * c->C;
    if (((uintptr_t)dev_samples & 15u) || bits_per_period % 128) return PCAL_ERR_ALIGNMENT;   // every period 16-byte aligned
    if (dev_out_folded && c->k_shift) return PCAL_ERR_STATE;
    c->stream = (cudaStream_t)cuda_stream;
    if (!c->prepared) c->first_bytes = bits_per_period / 8;
    const int rc = prepare(c);
    if (rc != PCAL_OK) return rc;
    c->started = true;
    const size_t nb = (size_t)c->n_bins * c->C;
    const uint8_t* p = reinterpret_cast<const uint8_t*>(dev_samples);
    // Small N_bins on the LUT path: the fold kernel of a period delivers T and the copy of P itself (one launch per
    // period, consecutive periods overlap); otherwise the DFT kernel and a device-to-device copy follow every period.
    const uint64_t piece = piece_samples(c, false);
    const bool fuse = can_fuse_dft(c) && !small_pieces() && n_per_period <= piece && bits_per_period >= 128;
    for (uint32_t k = 0; k < n_periods; ++k) {
        c->zero_pending = true;                       // the period's first post kernel overwrites the bins
        if (fuse) {
            c->fuse_req = true; c->fuse_out = nullptr;
            c->fuse_T_dev = reinterpret_cast<double2*>(dev_out_tones) + (size_t)k * nb;
            c->fuse_P_copy = dev_out_folded ? reinterpret_cast<double2*>(dev_out_folded) + (size_t)k * nb : nullptr;
        }
        int r = extract_segment(c, p + (size_t)k * (bits_per_period / 8), n_per_period);
        c->fuse_req = false; c->fuse_T_dev = nullptr; c->fuse_P_copy = nullptr;
        if (r != PCAL_OK) return r;
        if (fuse) continue;
        r = enqueue_dft(c, reinterpret_cast<double2*>(dev_out_tones) + (size_t)k * nb);
        if (r != PCAL_OK) return r;
        if (dev_out_folded)
            CU(cudaMemcpyAsync(dev_out_folded + (size_t)k * nb * 2, c->d_P, nb * sizeof(double2), cudaMemcpyDeviceToDevice, c->stream));
    }
    return PCAL_OK;
}

extern "C" int pcal_extract_host(pcal_ctx* c, const void* host_samples, uint64_t n_samples, void* cuda_stream) {
    if (!c) return PCAL_ERR_INVALID;
    if (n_samples == 0) return PCAL_OK;
    if (!host_samples) return PCAL_ERR_INVALID;
    if ((n_samples * (uint64_t)c->bits * c->C) % 8) return PCAL_ERR_ALIGNMENT;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!c->d_stage) CU(cudaMalloc(&c->d_stage, 2 * kStageBytes));
    const uint64_t total = n_samples * (uint64_t)c->bits * c->C / 8;
    const uint8_t* h = reinterpret_cast<const uint8_t*>(host_samples);
    const uint64_t bits_per_t = (uint64_t)c->bits * c->C;
    int buf = 0;
    for (uint64_t off = 0; off < total; off += kStageBytes, buf ^= 1) {
        const uint64_t bytes = total - off < kStageBytes ? total - off : kStageBytes;
        uint8_t* d = reinterpret_cast<uint8_t*>(c->d_stage) + (size_t)buf * kStageBytes;
        CU(cudaMemcpyAsync(d, h + off, bytes, cudaMemcpyHostToDevice, st));
        const bool promised = c->input_ready;
        c->input_ready = false;                        // the staging buffer is being written on this very stream
        const int r = pcal_extract(c, d, bytes * 8 / bits_per_t, st);
        c->input_ready = promised;
        if (r != PCAL_OK) return r;
    }
    CU(cudaStreamSynchronize(st));
    return PCAL_OK;
}

// The DFT kernel writes T both to d_T and, when `host_out` is device-visible pinned host memory
// (cudaHostAlloc / cudaHostRegister under unified addressing), straight into it: no copy node.
// outputs per warp of dft_kernel: as many as keep the grid at <= 32 CTAs, at most 4096 terms per warp
static uint32_t dft_opw(const pcal_ctx* c) {
    const uint32_t per_cta = kDftThreads / 32;
    uint32_t opw = 1;
    while ((uint64_t)c->C * ((c->n_bins + per_cta * opw - 1) / (per_cta * opw)) > 32 && (uint64_t)c->n_bins * opw * 2 <= 4096) opw *= 2;
    return opw;
}
static uint32_t dft_ctas(const pcal_ctx* c) {
    const uint32_t per_cta = kDftThreads / 32 * dft_opw(c);
    return (uint32_t)c->C * ((c->n_bins + per_cta - 1) / per_cta);
}

// stage C of the fold kernel can take the DFT itself: small N_bins, and C*N_bins complex values fit in its scratch
static bool can_fuse_dft(const pcal_ctx* c) {
    if (c->prepared && c->rot_eff == PCAL_ROT_GENERATOR && c->gen2) {
        if ((c->C > 4 && 4u * c->g2_ncls != (uint32_t)c->C) || c->g2_blocks > 1) return false;   // several launches per piece
        // two-stage DFT in the last CTA: cheap enough to sit in the serial final stage, and P and the scratch fit behind the
        // position sums in the kernel's rings (everything before its barriers and bookkeeping words)
        const uint32_t n1 = dft_n1_of(c->n_bins);
        const size_t ring = c->gen_smem - 1024;
        return (uint64_t)c->n_bins * (n1 + c->n_bins / n1) <= (1u << 17) &&
               2 * (size_t)c->n_bins * c->C * sizeof(double2) + 2 * kG2Fields * sizeof(long long) <= ring;
    }
    if (c->prepared && c->rot_eff == PCAL_ROT_GENERATOR) {
        if (!c->gen_fused) return false;
        // int8 / float32 generator kernels: the CTA that finishes last (pcal_gen_tail.cuh); bins, DFT scratch and the slice sums
        // of the reduction in the kernel's dynamic shared memory
        const uint32_t n1 = dft_n1_of(c->n_bins);
        return (uint64_t)c->n_bins * (n1 + c->n_bins / n1) <= (1u << 17) && (2 * (size_t)c->n_bins + 512) * sizeof(double2) <= c->gen_smem;
    }
    if (!(c->prepared && c->rot_eff == PCAL_ROT_LUT && c->fused)) return false;
    // the last finishing CTA of the fold kernel: two-stage DFT cheap enough for a serial stage, and 2 * C * N_bins complex
    // values (P and as much scratch) fit in the kernel's shared scratch (4096 / 2048 / 1024 doubles)
    const uint32_t n1 = dft_n1_of(c->n_bins);
    const uint32_t cap = c->kind == KIND_2BIT ? 2048u : 512u;
    return (uint64_t)c->n_bins * (n1 + c->n_bins / n1) <= (1u << 17) && 2u * c->n_bins * (uint32_t)c->C <= cap;
}

static int enqueue_dft(pcal_ctx* c, double2* second_dst) {
    const int rz = ensure_zeroed(c);
    if (rz != PCAL_OK) return rz;
    const size_t smem = 2 * (size_t)c->n_bins * sizeof(double2);
    const uint32_t opw = dft_opw(c), per_cta = kDftThreads / 32 * opw;
    launch_chain(dft_kernel, dim3((c->n_bins + per_cta - 1) / per_cta, c->C), kDftThreads, smem, c->stream,
                 (const double2*)c->d_P, (const double2*)c->d_W, c->d_T, second_dst, c->n_bins, (uint32_t)c->k_shift, opw,
                 (c->rot_eff == PCAL_ROT_LUT && c->fused) || (c->rot_eff == PCAL_ROT_GENERATOR && (c->gen2 || c->gen_fused)) ? c->d_tail_state : (TailState*)nullptr,
                 can_fuse_dft(c) ? 1 : 0);
    c->launches += 1;
    CU(cudaGetLastError());
    return PCAL_OK;
}

static double2* mapped_of(pcal_ctx* c, double* out);

extern "C" int pcal_finalize_async(pcal_ctx* c, double* out) {
    if (!c || !out) return PCAL_ERR_INVALID;
    double2* mapped = mapped_of(c, out);
    const int r = enqueue_dft(c, mapped);
    if (r != PCAL_OK) return r;
    if (!mapped)
        CU(cudaMemcpyAsync(out, c->d_T, (size_t)c->n_bins * c->C * sizeof(double2), cudaMemcpyDeviceToHost, c->stream));
    return PCAL_OK;
}

static double2* mapped_of(pcal_ctx* c, double* out) {
    if (out != c->last_out) {     // the attribute query costs more than a launch: remember the answer
        c->last_out = out; c->last_out_mapped = nullptr;
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, out) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer)
            c->last_out_mapped = reinterpret_cast<double2*>(at.devicePointer);
        cudaGetLastError();
    }
    return c->last_out_mapped;
}

extern "C" int pcal_integrate(pcal_ctx* c, const void* dev_samples, uint64_t n_samples, void* cuda_stream, double* out) {
    if (!c || !out) return PCAL_ERR_INVALID;
    int r = pcal_reset(c);
    if (r != PCAL_OK) return r;
    c->stream = (cudaStream_t)cuda_stream;
    if (!c->prepared) c->first_bytes = n_samples * (uint64_t)c->bits * c->C / 8;
    r = prepare(c);
    if (r != PCAL_OK) return r;
    // One launch for the whole period when the fold kernel can deliver T itself: a small DFT, the period is one
    // piece with at least one complete vector, and out is device-visible pinned memory.
    double2* mapped = mapped_of(c, out);
    const uint64_t piece = piece_samples(c, false);
    c->fuse_req = mapped && can_fuse_dft(c) && !small_pieces() && n_samples <= piece &&
                  n_samples * (uint64_t)c->bits * c->C / 8 >= 16 && dev_samples;
    c->fuse_out = mapped; c->fuse_T_dev = nullptr; c->fuse_P_copy = nullptr;
    r = pcal_extract(c, dev_samples, n_samples, cuda_stream);
    const bool fused_done = c->fuse_req;
    c->fuse_req = false;
    if (r != PCAL_OK) return r;
    c->stream = (cudaStream_t)cuda_stream;
    return fused_done ? PCAL_OK : pcal_finalize_async(c, out);
}

extern "C" int pcal_finalize(pcal_ctx* c, double* out) {
    if (!c || !out) return PCAL_ERR_INVALID;
    const int r = pcal_finalize_async(c, c->h_pinned);
    if (r != PCAL_OK) return r;
    CU(cudaStreamSynchronize(c->stream));
    memcpy(out, c->h_pinned, (size_t)c->n_bins * c->C * sizeof(double2));
    return PCAL_OK;
}

// PCal data analysis: DFT, then one analysis CTA per channel.
extern "C" int pcal_analyze(pcal_ctx* c, double* out_summary, double* out_bandpass) {
    if (!c || !out_summary) return PCAL_ERR_INVALID;
    const int r = enqueue_dft(c, nullptr);
    if (r != PCAL_OK) return r;
    AnalyzeParams ap;
    ap.P = c->d_P; ap.T = c->d_T; ap.summary = c->d_summary; ap.B = c->d_B;
    ap.f_s_hz = (double)c->Fs * 1e-6; ap.f_comb_hz = (double)c->Fcomb * 1e-6; ap.N = c->n_bins;
    ap.zero_offset_mask = 0;
    for (int i = 0; i < c->C; ++i) if (c->Foff[i] == 0) ap.zero_offset_mask |= 1u << i;
    const size_t smem = (size_t)c->n_bins * sizeof(double);
    analyze_kernel<<<c->C, kAnaThreads, smem, c->stream>>>(ap);
    c->launches += 1;
    CU(cudaGetLastError());
    const size_t sb = (size_t)c->C * kNSummary * sizeof(double), bb = (size_t)c->n_bins * c->C * sizeof(double2);
    CU(cudaMemcpyAsync(c->h_ana, c->d_summary, sb, cudaMemcpyDeviceToHost, c->stream));
    if (out_bandpass) CU(cudaMemcpyAsync(reinterpret_cast<char*>(c->h_ana) + sb, c->d_B, bb, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    memcpy(out_summary, c->h_ana, sb);
    if (out_bandpass) memcpy(out_bandpass, reinterpret_cast<char*>(c->h_ana) + sb, bb);
    return PCAL_OK;
}

// ---- multi-pass counter-rotation (R27) ----------------------------------------------
static int residual_rotation_of(pcal_ctx* c, const double* dev_series, uint32_t n_periods, uint32_t zero_mask, double* out) {
    double* d_out = c->d_summary;       // [C][kNSummary] >= [C][kNResidual]
    residual_rotation_kernel<<<c->C, kAnaThreads, 0, c->stream>>>(reinterpret_cast<const double2*>(dev_series), n_periods, c->n_bins,
                                                                   (uint32_t)c->C, zero_mask, d_out);
    c->launches += 1;
    CU(cudaGetLastError());
    const size_t bytes = (size_t)c->C * kNResidual * sizeof(double);
    CU(cudaMemcpyAsync(c->h_ana, d_out, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    memcpy(out, c->h_ana, bytes);
    return PCAL_OK;
}

extern "C" int pcal_residual_rotation(pcal_ctx* c, const double* dev_series_tones, uint32_t n_periods, double* out) {
    if (!c || !dev_series_tones || !out || n_periods == 0) return PCAL_ERR_INVALID;
    uint32_t zero_mask = 0;
    for (int i = 0; i < c->C; ++i) if (c->Foff[i] == 0) zero_mask |= 1u << i;
    return residual_rotation_of(c, dev_series_tones, n_periods, zero_mask, out);
}

extern "C" int pcal_refine_offset(pcal_ctx* c, const void* dev_samples, uint64_t n_per_period, uint32_t n_periods, void* cuda_stream,
                                  uint32_t max_passes, double tol_rad, double* out_f, double* out_history, uint32_t* out_passes) {
    if (!c || !dev_samples || !out_f || n_per_period == 0 || n_periods < 2 || max_passes == 0 || !(tol_rad >= 0)) return PCAL_ERR_INVALID;
    if (c->C != 1) return PCAL_ERR_UNSUPPORTED;
    const double fs = (double)c->Fs * 1e-6, fcomb = (double)c->Fcomb * 1e-6;
    const double t_int = (double)n_per_period / fs;
    const uint32_t zero_mask = c->Foff[0] == 0 ? 1u : 0u;    // the band is fixed by the starting offset (tone 0 is sin(0) there)
    double f = (double)c->Foff[0] * 1e-6;
    double2* d_series = nullptr;
    CU(cudaMalloc(&d_series, (size_t)n_periods * c->n_bins * sizeof(double2)));
    int rc = PCAL_OK;
    uint32_t passes = 0;
    for (uint32_t k = 0; k < max_passes && rc == PCAL_OK; ++k) {
        pcal_ctx* p = nullptr;        // one context per pass: the rotator (table or generator) of this pass's frequency
        rc = pcal_create(&p, fs, fcomb, f, c->bits, c->enc, 1);
        if (rc == PCAL_OK) rc = pcal_set_rotator(p, c->rot_req);
        if (rc == PCAL_OK) rc = pcal_extract_series(p, dev_samples, n_per_period, n_periods, cuda_stream, reinterpret_cast<double*>(d_series), nullptr);
        double res[kNResidual] = {0.0, 0.0, 0.0};
        if (rc == PCAL_OK) rc = residual_rotation_of(p, reinterpret_cast<const double*>(d_series), n_periods, zero_mask, res);
        pcal_destroy(p);
        if (rc != PCAL_OK) break;
        passes = k + 1;
        if (out_history) { out_history[4 * k] = f; out_history[4 * k + 1] = res[0]; out_history[4 * k + 2] = res[1]; out_history[4 * k + 3] = res[2]; }
        if (fabs(res[0]) <= tol_rad) break;
        const double fn = (double)llround((f + res[0] / (2.0 * M_PI * t_int)) * 1e6) * 1e-6;     // counter-rotate, 1 uHz grid
        if (!(fn >= 0.0) || !(fn < fs)) { rc = PCAL_ERR_INVALID; break; }
        f = fn;
    }
    cudaFree(d_series);
    if (rc != PCAL_OK) return rc;
    *out_f = f;
    if (out_passes) *out_passes = passes;
    pcal_reset(c);                    // started = false: the offset may be replaced
    return pcal_set_channel_offsets(c, &f);
}

// exp(+-j 2 pi k b / N) applied on the host to (un)shift the folded period
static void kshift_bins(const pcal_ctx* c, double* bins, int sign) {
    if (!c->k_shift) return;
    for (int ch = 0; ch < c->C; ++ch)
        for (uint32_t b = 0; b < c->n_bins; ++b) {
            const uint64_t k = ((uint64_t)c->k_shift * b) % c->n_bins;
            const long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)c->n_bins;
            const long double cs = cosl(ang), sn = sign * sinl(ang);
            double* z = bins + ((size_t)ch * c->n_bins + b) * 2;
            const long double re = z[0] * cs - z[1] * sn, im = z[0] * sn + z[1] * cs;
            z[0] = (double)re; z[1] = (double)im;
        }
}

// the exact integer bins, where the context keeps them (integer samples, no rotation): the exchange calls maintain them too
static long long* exact_bins_of(const pcal_ctx* c) {
    if (c->kind == KIND_F32 || c->k_shift) return nullptr;
    for (int i = 0; i < c->C; ++i) if (c->Foff[i]) return nullptr;
    return c->d_Pint;
}

extern "C" int pcal_get_folded(pcal_ctx* c, double* out) {
    if (!c || !out) return PCAL_ERR_INVALID;
    { const int rz = ensure_zeroed(c); if (rz != PCAL_OK) return rz; }
    const size_t bytes = (size_t)c->n_bins * c->C * sizeof(double2);
    CU(cudaMemcpyAsync(c->h_pinned, c->d_P, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    memcpy(out, c->h_pinned, bytes);
    kshift_bins(c, out, +1);
    return PCAL_OK;
}

extern "C" int pcal_get_folded_i64(pcal_ctx* c, int64_t* out) {
    if (!c || !out) return PCAL_ERR_INVALID;
    if (c->kind == KIND_F32 || c->k_shift) return PCAL_ERR_STATE;
    for (int i = 0; i < c->C; ++i) if (c->Foff[i]) return PCAL_ERR_STATE;
    { const int rz = ensure_zeroed(c); if (rz != PCAL_OK) return rz; }
    const size_t bytes = (size_t)c->n_bins * c->C * sizeof(long long);
    CU(cudaMemcpyAsync(c->h_pinned, c->d_Pint, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    memcpy(out, c->h_pinned, bytes);
    return PCAL_OK;
}

extern "C" int pcal_add_folded(pcal_ctx* c, const double* bins) {
    if (!c || !bins) return PCAL_ERR_INVALID;
    { const int rz = ensure_zeroed(c); if (rz != PCAL_OK) return rz; }
    const uint32_t n = c->n_bins * (uint32_t)c->C;
    CU(cudaStreamSynchronize(c->stream));
    memcpy(c->h_pinned, bins, (size_t)n * sizeof(double2));
    kshift_bins(c, c->h_pinned, -1);
    CU(cudaMemcpyAsync(c->d_tmp, c->h_pinned, (size_t)n * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
    add_bins_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(c->d_P, exact_bins_of(c), c->d_tmp, n);
    c->launches += 1;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(c->stream));
    return PCAL_OK;
}

extern "C" int pcal_reset(pcal_ctx* c) {
    if (!c) return PCAL_ERR_INVALID;
    c->zero_pending = true;   // the next post kernel overwrites; other readers zero first
    c->n_processed = 0;
    c->started = false;
    return PCAL_OK;
}

extern "C" int pcal_get_folded_dev(pcal_ctx* c, double* dev_bins) {
    if (!c || !dev_bins) return PCAL_ERR_INVALID;
    { const int rz = ensure_zeroed(c); if (rz != PCAL_OK) return rz; }
    CU(cudaMemcpyAsync(dev_bins, c->d_P, (size_t)c->n_bins * c->C * sizeof(double2), cudaMemcpyDeviceToDevice, c->stream));
    return PCAL_OK;
}

extern "C" int pcal_add_folded_dev(pcal_ctx* c, const double* dev_bins) {
    if (!c || !dev_bins) return PCAL_ERR_INVALID;
    { const int rz = ensure_zeroed(c); if (rz != PCAL_OK) return rz; }
    const uint32_t n = c->n_bins * (uint32_t)c->C;
    add_bins_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(c->d_P, exact_bins_of(c), reinterpret_cast<const double2*>(dev_bins), n);
    c->launches += 1;
    CU(cudaGetLastError());
    return PCAL_OK;
}

extern "C" int pcal_set_folded_sum_dev(pcal_ctx* c, const double* dev_parts, uint32_t n_parts) {
    if (!c || !dev_parts || n_parts == 0) return PCAL_ERR_INVALID;
    const uint32_t n = c->n_bins * (uint32_t)c->C;
    sum_parts_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(c->d_P, exact_bins_of(c), reinterpret_cast<const double2*>(dev_parts), n, n_parts);
    c->launches += 1;
    CU(cudaGetLastError());
    c->zero_pending = false;      // the accumulators now hold exactly the sum
    return PCAL_OK;
}

// The exchange step of a time-sharded SERIES in one go: n_periods folded periods per rank were gathered into dev_parts
// ([n_parts][n_periods][C][N_bins] complex); each period's bins are added in rank order, then its DFT is taken.
extern "C" int pcal_finalize_series_sum_dev(pcal_ctx* c, const double* dev_parts, uint32_t n_parts, uint32_t n_periods,
                                            double* dev_out_folded, double* dev_out_tones) {
    if (!c || !dev_parts || !dev_out_folded || !dev_out_tones || n_parts == 0) return PCAL_ERR_INVALID;
    if (n_periods == 0) return PCAL_OK;
    const uint64_t n64 = (uint64_t)c->n_bins * c->C * n_periods;
    if (n64 > (1ull << 30) || (uint64_t)c->C * n_periods > 65535) return PCAL_ERR_INVALID;
    const uint32_t n = (uint32_t)n64;
    sum_parts_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(reinterpret_cast<double2*>(dev_out_folded), (long long*)nullptr,
                                                             reinterpret_cast<const double2*>(dev_parts), n, n_parts);
    // one DFT grid over (period, channel) rows: the series is laid out [period][channel][bin]
    const size_t smem = 2 * (size_t)c->n_bins * sizeof(double2);
    const uint32_t per_cta = kDftThreads / 32;
    dft_kernel<<<dim3((c->n_bins + per_cta - 1) / per_cta, c->C * n_periods), kDftThreads, smem, c->stream>>>(
        reinterpret_cast<const double2*>(dev_out_folded), (const double2*)c->d_W, reinterpret_cast<double2*>(dev_out_tones),
        (double2*)nullptr, c->n_bins, (uint32_t)c->k_shift, 1u, (TailState*)nullptr, 0);
    c->launches += 2;
    CU(cudaGetLastError());
    return PCAL_OK;
}

// Generator accuracy study: one device thread per case.
extern "C" int pcal_generator_study(const pcal_gen_case_t* cases, uint32_t n_cases, uint64_t n_steps, uint32_t n_chk,
                                    double* out_err) {
    if (!cases || !out_err || n_cases == 0 || n_chk == 0 || n_steps == 0 || n_steps >= (1ull << 40)) return PCAL_ERR_INVALID;
    std::vector<GenStudyCase> h(n_cases);
    for (uint32_t i = 0; i < n_cases; ++i) {
        const pcal_gen_case_t& u = cases[i];
        if (u.form < PCAL_GEN_CFO || u.form > PCAL_GEN_DIRECT || (u.precision != 32 && u.precision != 64)) return PCAL_ERR_INVALID;
        if (!(u.f_s_hz > 0) || !(u.f_rot_hz >= 0) || !(u.f_rot_hz < u.f_s_hz)) return PCAL_ERR_INVALID;
        GenStudyCase& g = h[i];
        g.form = u.form; g.precision = u.precision; g.Fs = to_uhz(u.f_s_hz); g.F = to_uhz(u.f_rot_hz);
        if (g.Fs == 0 || g.Fs >= (1ull << 61)) return PCAL_ERR_INVALID;
        const double dphi = 2.0 * M_PI * (double)g.F / (double)g.Fs;         // eq. 2.5
        g.cn = cos(dphi); g.sn = sin(dphi); g.eps = 2.0 * sin(0.5 * dphi); g.two_c = 2.0 * cos(dphi);
        g.s_half = sin(0.5 * dphi); g.dphi32 = (float)dphi;
    }
    GenStudyCase* d_cases = nullptr;
    double* d_err = nullptr;
    const size_t eb = (size_t)n_cases * n_chk * sizeof(double);
    if (cudaMalloc(&d_cases, n_cases * sizeof(GenStudyCase)) != cudaSuccess || cudaMalloc(&d_err, eb) != cudaSuccess) {
        cudaFree(d_cases); cudaGetLastError(); return PCAL_ERR_DEVICE;
    }
    int rc = PCAL_OK;
    if (cudaMemcpy(d_cases, h.data(), n_cases * sizeof(GenStudyCase), cudaMemcpyHostToDevice) != cudaSuccess) rc = PCAL_ERR_DEVICE;
    if (rc == PCAL_OK) {
        gen_study_kernel<<<(n_cases + 31) / 32, 32>>>(d_cases, n_cases, n_steps, n_chk, d_err);
        if (cudaGetLastError() != cudaSuccess || cudaMemcpy(out_err, d_err, eb, cudaMemcpyDeviceToHost) != cudaSuccess) rc = PCAL_ERR_DEVICE;
    }
    cudaFree(d_cases); cudaFree(d_err); cudaGetLastError();
    return rc;
}

// ---------------------------------------------------------------------------------------------
// pcal_fold_noalloc (include/pcal_noalloc.h): rotate + fold one segment without allocating anything.
// gen_kernel and post_gen_kernel as they are; their scratch -- the per-CTA partial bins -- is this file-scope array
// instead of cudaMalloc'd memory.  Every device that loads the library holds its 2.5 MiB until the process exits.
// In HOST code the name of a __device__ array is a host-side stand-in, not a device address: the kernels get the
// address that cudaGetSymbolAddress returns for the current device (looked up once per device, below).
// Shared by every call on the device, never cleared: gen_kernel writes all n_bins partial bins of each of its CTAs
// before post_gen_kernel reads exactly those; calls that overlap on the GPU race on it (pcal_noalloc.h).
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[PCAL_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int kNoAllocMaxDevices = 64;
struct NoAllocDevice {
    bool ready;
    double2* scratch;      // device address of g_noalloc_scratch on this device
    int sm_count;
};
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];
std::mutex g_noalloc_mutex;

// once per device, with that device current: address of the scratch array, SM count, shared-memory attribute of the kernels
int noalloc_setup(int dev, NoAllocDevice** out) {
    if (dev < 0 || dev >= kNoAllocMaxDevices) return PCAL_ERR_DEVICE;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoAllocDevice& d = g_noalloc_dev[dev];
    if (!d.ready) {
        void* ptr = nullptr;
        CU(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
        if (!ptr || ((uintptr_t)ptr & 255u)) return PCAL_ERR_DEVICE;
        CU(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaFuncSetAttribute(gen_kernel<KIND_2BIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gen_smem_bytes<KIND_2BIT>()));
        CU(cudaFuncSetAttribute(gen_kernel<KIND_I8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gen_smem_bytes<KIND_I8>()));
        CU(cudaFuncSetAttribute(gen_kernel<KIND_F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gen_smem_bytes<KIND_F32>()));
        d.scratch = reinterpret_cast<double2*>(ptr);
        d.ready = true;
    }
    *out = &d;
    return PCAL_OK;
}
}  // namespace

extern "C" int pcal_fold_noalloc(const void* dev_samples, uint64_t n_samples, uint64_t start_index, double f_s_hz, double f_comb_hz,
                                 double f_offset_hz, int bits, int encoding, int accumulate, double* dev_out_bins, void* cuda_stream) {
    if (!dev_out_bins || (!dev_samples && n_samples)) return PCAL_ERR_INVALID;
    if (!(f_s_hz > 0) || !(f_comb_hz > 0) || !(f_offset_hz >= 0) || !(f_offset_hz < f_s_hz)) return PCAL_ERR_INVALID;
    const uint64_t Fs = to_uhz(f_s_hz), Fc = to_uhz(f_comb_hz), Fo = to_uhz(f_offset_hz);
    if (Fs == 0 || Fc == 0 || Fs % Fc != 0 || Fs / Fc < 2 || Fs >= (1ull << 62)) return PCAL_ERR_INVALID;
    int kind;
    if (bits == 2 && (encoding == PCAL_ENC_OFFSET_BINARY || encoding == PCAL_ENC_SIGN_MAG)) kind = KIND_2BIT;
    else if (bits == 8 && encoding == PCAL_ENC_TWOS_COMPLEMENT) kind = KIND_I8;
    else if (bits == 32 && encoding == PCAL_ENC_IEEE_FLOAT) kind = KIND_F32;
    else return PCAL_ERR_INVALID;
    if (Fs / Fc > PCAL_NOALLOC_MAX_BINS) return PCAL_ERR_LIMIT;          // the scratch array holds 160 x 1024 bins
    const uint32_t n_bins = (uint32_t)(Fs / Fc);
    if (((uintptr_t)dev_samples & 15u) || ((uintptr_t)dev_out_bins & 15u) || (n_samples * (uint64_t)bits) % 8u) return PCAL_ERR_ALIGNMENT;
    // a CTA iteration of gen_kernel: the largest multiple of lcm(N_bins, samples per load) that 256 loads hold
    const uint32_t spt = kind == KIND_F32 ? 4u : 16u;
    const uint64_t unit = lcm_sat(n_bins, spt, 1u << 20), cap = (uint64_t)kThreads * spt;
    if (unit > cap) return PCAL_ERR_UNSUPPORTED;
    const uint32_t span = (uint32_t)(unit * (cap / unit));

    int dev = 0;
    CU(cudaGetDevice(&dev));
    NoAllocDevice* nd = nullptr;
    const int rc = noalloc_setup(dev, &nd);
    if (rc != PCAL_OK) return rc;
    const uint32_t grid = (uint32_t)nd->sm_count < PCAL_NOALLOC_MAX_CTAS ? (uint32_t)nd->sm_count : PCAL_NOALLOC_MAX_CTAS;
    if ((size_t)grid * n_bins * sizeof(double2) > PCAL_NOALLOC_SCRATCH_BYTES) return PCAL_ERR_LIMIT;     // (cannot happen: both capped above)
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint8_t* data = reinterpret_cast<const uint8_t*>(dev_samples);
    const uint64_t load_bytes = kind == KIND_2BIT ? 4 : 16;
    const uint64_t tile = (uint64_t)(kTileSamples / (kThreads * spt)) * span;          // samples per tile of a CTA
    const uint64_t piece = (uint64_t)(small_pieces() ? 2 : kGenMaxTiles) * grid * tile;   // the resync table of a CTA holds 256 tiles (PCAL_SMALL_PIECES: tests)
    uint64_t done = 0;
    bool first = true;
    do {
        const uint64_t n = n_samples - done < piece ? n_samples - done : piece;
        const uint8_t* base = data + done * (uint64_t)bits / 8;
        const uint64_t n0 = start_index + done;
        const uint64_t n_loads = n * (uint64_t)bits / 8 / load_bytes;
        if (n_loads) {
            GenParams gp;
            memset(&gp, 0, sizeof(gp));
            gp.data = base; gp.n_loads = n_loads; gp.span = span;
            gp.n_tiles = (n_loads * spt + tile - 1) / tile;
            gp.n_iters = (n_loads * spt + span - 1) / span;
            gp.Fs = Fs; gp.Foff = Fo;
            gp.k0 = mulmod_host(n0 % Fs, Fo, Fs);
            gp.rho = phasor_neg_host(mulmod_host(span, Fo, Fs), Fs);
            gp.rho2 = phasor_neg_host(mulmod_host(2ull * span, Fo, Fs), Fs);
            for (uint32_t k = 0; k < 16; ++k) gp.tw[k] = phasor_neg_host(mulmod_host(k, Fo, Fs), Fs);
            gp.n_bins = n_bins; gp.sign_mag = encoding == PCAL_ENC_SIGN_MAG;
            gp.dec_mask = 0x00600000u; gp.dec_one = 0x3F800000u;
            gp.input_ready = 0;                       // the samples may come from earlier work on the stream
            gp.tail.st = nullptr;                     // no fused tail: partial bins of CTA i at scratch + i * n_bins
            gp.tail.partial = nd->scratch;
            if (kind == KIND_2BIT) launch_chain(gen_kernel<KIND_2BIT>, grid, kThreads, gen_smem_bytes<KIND_2BIT>(), st, gp);
            else if (kind == KIND_I8) launch_chain(gen_kernel<KIND_I8>, grid, kThreads, gen_smem_bytes<KIND_I8>(), st, gp);
            else launch_chain(gen_kernel<KIND_F32>, grid, kThreads, gen_smem_bytes<KIND_F32>(), st, gp);
        }
        GenPostParams gr;
        memset(&gr, 0, sizeof(gr));
        gr.partial = nd->scratch; gr.P = reinterpret_cast<double2*>(dev_out_bins);
        gr.tail = base + n_loads * load_bytes;
        gr.n0 = n0; gr.n_done = n_loads * spt; gr.n_total = n; gr.Fs = Fs; gr.Foff = Fo;
        gr.grid = n_loads ? grid : 0; gr.n_bins = n_bins; gr.kind = kind; gr.sign_mag = encoding == PCAL_ENC_SIGN_MAG;
        gr.overwrite = (first && !accumulate) ? 1 : 0;
        if (n || gr.overwrite) launch_chain(post_gen_kernel, (n_bins + 31) / 32, kPostThreads, 0, st, gr);
        first = false;
        done += n;
    } while (done < n_samples);
    CU(cudaGetLastError());
    return PCAL_OK;
}
