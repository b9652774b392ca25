/*
 * pcal_probe.h -- measurement hooks of libpcal.  NOT part of the extraction API (include/pcal.h): these calls exist for
 * bench.py's roofline report ("pipe peaks ... are to be measured on the box"; "CUDA events around
 * pcal_extract only") and compute nothing a user of the library needs.
 */
#ifndef PCAL_PROBE_H_
#define PCAL_PROBE_H_

#include "pcal.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Timing hook: when enabled, every launch of the hot kernel (the fused load/decode/fold kernel of the LUT path or the
 * generator kernel) is bracketed by CUDA events on the launching stream.  pcal_get_profile synchronises the stream and
 * returns the summed event time in milliseconds and the number of hot-kernel launches since profiling was enabled (or
 * since the last pcal_get_profile).  Bracketing serialises consecutive launches: what it measures is the latency of an
 * isolated launch, not its cost in a pipelined series. */
int pcal_set_profiling(pcal_ctx *ctx, int enable);
int pcal_get_profile(pcal_ctx *ctx, double *hot_kernel_ms, uint64_t *hot_kernel_launches);

/* Calibration: enqueue a pure streaming read (no decode, no fold) of n_bytes from dev ([device], 16-byte aligned) on
 * cuda_stream, with the load instruction, block size and pipelining of the fold kernels; consecutive probes may overlap
 * (programmatic dependent launch), like consecutive fold kernels.  Asynchronous; computes nothing; the caller times it.
 * What it reaches on a given size is the practical ceiling of a read-once kernel of that size. */
int pcal_read_probe(pcal_ctx *ctx, const void *dev, uint64_t n_bytes, void *cuda_stream);

/* Calibration: the measured issue rate of one pipe of the current device.  kind 0 = FFMA (fp32 FMA pipe), 1 = LOP3
 * (integer/logic pipe), 2 = IMMA m16n8k16 s8, 3 = IMMA m16n8k32 u8 x s8 (the legacy tensor path of the generator kernels: int8 / 2-bit).
 * out_per_s [host]: thread-instructions per second (kind 0, 1) or warp-level MMA instructions per second (kind 2, 3) with
 * every SM busy.
 * Synchronous, default stream, no context needed. */
int pcal_pipe_probe(int kind, double *out_per_s);

#ifdef __cplusplus
}
#endif
#endif /* PCAL_PROBE_H_ */
