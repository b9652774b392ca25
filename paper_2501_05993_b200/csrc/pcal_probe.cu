// pcal_probe.cu -- the measurement hooks of include/pcal_probe.h: calibration kernels (a pure streaming read, issue-rate
// loops) and the event bracket around the hot kernel.  They serve bench.py's roofline report, not the extraction path.
#include <stdlib.h>
#include <string.h>

#include "../../include/pcal_probe.h"
#include "pcal_ctx.h"

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
// gen_mma_kernel), 3: IMMA m16n8k32 u8 x s8 (gen2_kernel).  Eight independent dependency chains per thread, `iters` trips; the result is written so that
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
            else if (KIND_P == 2) asm volatile("mma.sync.aligned.m16n8k16.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
                              : "+r"(d[j][0]), "+r"(d[j][1]), "+r"(d[j][2]), "+r"(d[j][3]) : "r"(x), "r"(y), "r"(a[j]));
            else asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                              : "+r"(d[j][0]), "+r"(d[j][1]), "+r"(d[j][2]), "+r"(d[j][3]) : "r"(x), "r"(y), "r"(x ^ y), "r"(y + 1u), "r"(a[j]), "r"(a[j] ^ x));
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j] + __float_as_uint(f[j]) + (uint32_t)(d[j][0] + d[j][1] + d[j][2] + d[j][3]);
    if (s == 0x5ca1ab1eu) out[0] = s;
}

}  // namespace pcal

using namespace pcal;

extern "C" int pcal_read_probe(pcal_ctx* c, const void* dev, uint64_t n_bytes, void* cuda_stream) {
    if (!c || !dev) return PCAL_ERR_INVALID;
    if ((uintptr_t)dev & 15u) return PCAL_ERR_ALIGNMENT;
    int occ = occupancy_of(read_probe_kernel, 0);
    if (occ < 1) return PCAL_ERR_DEVICE;
    uint32_t grid = (uint32_t)(c->sm_count * occ);
    if (const char* g = getenv("PCAL_PROBE_GRID")) grid = (uint32_t)atoi(g);      // tuning runs only
    const char* pp = getenv("PCAL_PROBE_PDL");
    if (!(pp && pp[0] == '0'))      // default: consecutive probes may overlap, like the fold kernels
        launch_chain(read_probe_kernel, grid, kThreads, 0, (cudaStream_t)cuda_stream,
                     reinterpret_cast<const uint4*>(dev), (uint64_t)(n_bytes / 16), reinterpret_cast<uint32_t*>(c->d_tmp));
    else
        read_probe_kernel<<<grid, kThreads, 0, (cudaStream_t)cuda_stream>>>(
            reinterpret_cast<const uint4*>(dev), n_bytes / 16, reinterpret_cast<uint32_t*>(c->d_tmp));
    c->launches += 1;
    CU(cudaGetLastError());
    return PCAL_OK;
}

extern "C" int pcal_pipe_probe(int kind, double* out_per_s) {
    if (!out_per_s || kind < 0 || kind > 3) return PCAL_ERR_INVALID;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    uint32_t* d_out = nullptr;
    CU(cudaMalloc(&d_out, sizeof(uint32_t)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const uint32_t iters = 4096, grid = (uint32_t)sms * 8;       // 8 CTAs of 256 threads per SM: every scheduler has 16 warps
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        if (kind == 0) pipe_probe_kernel<0><<<grid, kThreads>>>(iters, d_out);
        else if (kind == 1) pipe_probe_kernel<1><<<grid, kThreads>>>(iters, d_out);
        else if (kind == 2) pipe_probe_kernel<2><<<grid, kThreads>>>(iters, d_out);
        else pipe_probe_kernel<3><<<grid, kThreads>>>(iters, d_out);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    if (cudaGetLastError() != cudaSuccess || !(best < 1e29f)) return PCAL_ERR_DEVICE;
    const double per_thread = (double)iters * 8.0, threads = (double)grid * kThreads;
    *out_per_s = (kind >= 2 ? per_thread * threads / 32.0 : per_thread * threads) / (best * 1e-3);
    return PCAL_OK;
}

extern "C" int pcal_set_profiling(pcal_ctx* c, int enable) {
    if (!c) return PCAL_ERR_INVALID;
    CU(cudaStreamSynchronize(c->stream));
    prof_collect(c);
    c->profiling = enable != 0;
    c->prof_ms = 0.0; c->prof_launches = 0;
    return PCAL_OK;
}

extern "C" int pcal_get_profile(pcal_ctx* c, double* ms, uint64_t* launches) {
    if (!c || !ms || !launches) return PCAL_ERR_INVALID;
    CU(cudaStreamSynchronize(c->stream));
    prof_collect(c);
    *ms = c->prof_ms; *launches = c->prof_launches;
    c->prof_ms = 0.0; c->prof_launches = 0;
    return PCAL_OK;
}
