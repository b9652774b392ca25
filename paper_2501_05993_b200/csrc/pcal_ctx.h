// pcal_ctx.h -- internal to libpcal: the context behind the opaque pcal_ctx of include/pcal.h and the launch helpers
// shared by pcal_api.cu (the product calls) and pcal_probe.cu (the measurement hooks of include/pcal_probe.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/pcal.h"
#include "pcal_common.cuh"

namespace pcal { struct FoldParams; struct TailState; }    // (pcal_fold.cuh, pcal_post.cuh: kernels live in pcal_api.cu only)

struct pcal_ctx {
    // problem
    uint64_t Fs, Fcomb, Foff[PCAL_MAX_CHANNELS], Feff[PCAL_MAX_CHANNELS];
    int bits, enc, C, kind, sign_mag;
    uint32_t n_bins;
    int rot_req, rot_eff, k_shift;
    uint64_t n_processed;
    bool started, prepared, all_zero;
    // LUT-mode geometry
    uint32_t spv, F, q, R, grid;
    uint64_t M, nrot[PCAL_MAX_CHANNELS], lut_len[PCAL_MAX_CHANNELS];
    uint32_t lut_off_h[PCAL_MAX_CHANNELS];   // first table entry of every channel (host copy)
    // generator-mode geometry
    uint32_t gen_grid, gen_spt, gen_span;   // (gen_span: samples per CTA iteration of the FFMA2 kernel, a multiple of N_bins)
    bool gen_mma;                   // int8 samples, N_bins | 2048: tensor-core generator kernel (pcal_gen_mma.cuh)
    bool gen_fused;                 // int8 / float32 generator kernels: reduction, tail and DFT by their last CTAs (pcal_gen_tail.cuh)
    bool gen2;                      // 2-bit samples: warp-specialised tensor-core generator kernel (pcal_gen2.cuh)
    uint32_t g2_span_t, g2_chunks;  // ... its row: time samples, 16-byte chunks
    uint32_t g2_cpw, g2_rt;         // ... chunks per consumer warp (1, 2, 4), rows per tile (128, 64, 32)
    uint32_t g2_blocks;             // ... column blocks of a row (rows longer than 32 chunks are served 32 chunks per launch)
    uint32_t g2_ncls;               // ... byte classes (four channels each) of 8 / 16-channel words served by one launch (1, 2, 4)
    double2 *d_g2_rtab, *d_g2_tw;   // ... stride phasors [C][32], position factors [C][span_t]
    uint32_t* d_g2_ctr;             // ... [slot][2] batch and arrival counters
    long long* d_g2_posacc;         // ... [slot][2*2048] exact per-position sums
    size_t gen_smem;
    // device
    int device, sm_count;
    cudaStream_t stream;
    double2 *d_P, *d_T, *d_W, *d_lut, *d_gen_partial, *d_tmp;
    long long* d_Pint;
    uint32_t *d_lut_off, *d_lut_len;
    void *d_partial, *d_stage;
    double* d_val;                  // [q][F][32] replica sums (stage 1 of pcal_post.cuh)
    bool fused;                     // reduction + rotation run inside the fold kernel (pcal_tail.cuh)
    uint32_t* d_cnt;                // [slot][q+1] arrival counters of the fused tail
    double2* d_G;                   // [slot][q][C*n_bins] per-group bins of the fused tail
    pcal::TailState* d_tail_state;        // tickets and progress counters of the fused tail
    size_t partial_slot_bytes;
    uint32_t tail_tpp;              // threads per (channel, bin) pair in stage B of the fused tail
    uint32_t rot_tpp;               // threads per (channel, bin) pair in rotate_fold_kernel
    uint64_t first_bytes;           // bytes of the first segment / period seen before the geometry was fixed (prepare): a size hint
    bool input_ready;               // pcal_set_input_ready: sample buffers are complete when extract is called
    bool zero_pending;              // reset happened, accumulators not yet overwritten or zeroed
    double* h_pinned;
    double2* fuse_out;              // pcal_integrate: the fold kernel of this call also takes the DFT and writes T here (or null)
    double2 *fuse_T_dev, *fuse_P_copy;   // pcal_extract_series: device destinations of T and of a copy of P for the piece being enqueued
    bool fuse_req;                  // ... requested for the piece being enqueued
    const double* last_out;         // pcal_finalize_async: last host buffer seen and its device mapping (or null)
    double2* last_out_mapped;
    double *d_summary, *h_ana;      // analysis outputs: [C][8] + band-pass [C][N] complex
    double2* d_B;
    uint64_t launches;
    void (*fold2)(const pcal::FoldParams);      // the fold_2bit_kernel instantiation in use
    // profiling hook
    bool profiling;
    std::vector<cudaEvent_t>* ev;   // pairs (start, stop) recorded so far
    size_t ev_used;
    double prof_ms;
    uint64_t prof_launches;
};

// bracket the hot kernel with events on the launching stream (only when profiling is on)
static inline void prof_mark(pcal_ctx* c, cudaStream_t st) {
    if (!c->profiling) return;
    if (!c->ev) c->ev = new std::vector<cudaEvent_t>();
    if (c->ev_used == c->ev->size()) { cudaEvent_t e; cudaEventCreate(&e); c->ev->push_back(e); }
    cudaEventRecord((*c->ev)[c->ev_used++], st);
}
static inline void prof_collect(pcal_ctx* c) {
    for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, (*c->ev)[i], (*c->ev)[i + 1]) == cudaSuccess) { c->prof_ms += ms; c->prof_launches++; }
    }
    c->ev_used = 0;
    cudaGetLastError();
}

// Programmatic dependent launch: the kernels of one step form a chain; each is launched with
// programmatic stream serialization so that its CTAs can be scheduled while its predecessor is still
// running (hiding the launch latency), and each starts with griddepcontrol.wait (pdl_wait_release in
// pcal_common.cuh), i.e. touches memory only after the predecessor has completed and flushed.
// PCAL_NO_PDL=1 falls back to plain stream order.
static inline bool use_pdl() {
    static const bool on = [] { const char* e = getenv("PCAL_NO_PDL"); return !(e && e[0] == '1'); }();
    return on;
}
template <typename... KArgs, typename... Args>
static void launch_chain(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = use_pdl() ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, args...);
}

#define CU(x) do { if ((x) != cudaSuccess) { cudaGetLastError(); return PCAL_ERR_DEVICE; } } while (0)


template <typename K>
static inline int occupancy_of(K kernel, size_t smem) {
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, pcal::kThreads, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    return occ;
}

