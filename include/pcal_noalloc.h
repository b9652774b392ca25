/*
 * pcal_noalloc.h -- ONE entry point of libpcal that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it -- and every other path of this library works on a context whose buffers pcal_create / the first pcal_extract
 * allocate.  pcal_fold_noalloc rotates and folds one segment of a single-channel stream (eq. 2.3 + eq. 2.2,
 * PAPER.md:44-57) with the generator kernel of the float32 path (`gen_kernel`, pcal_gen.cuh: eq. 2.5-2.9, a
 * coupled-form oscillator re-seeded from the exactly reduced integer phase at least every 2^16 samples) followed by
 * `post_gen_kernel` (deterministic reduction of the per-CTA partial bins, ragged tail with exact phases), i.e. steps
 * a1-a5 of the hot path; the N_bins-point DFT (a6) is left to the caller.  The kernels are the library's own,
 * unchanged; what differs is where their scratch -- the per-CTA partial bins -- lives: not in memory obtained with
 * cudaMalloc but in a file-scope `static __device__` array of the library.
 *
 * The limit: that array is 160 CTAs x 1024 bins x 16 bytes = 2.5 MiB (PCAL_NOALLOC_SCRATCH_BYTES), held by every GPU
 * that loads the library until the process exits.  Hence N_bins = f_s / f_comb <= PCAL_NOALLOC_MAX_BINS (1024), one
 * channel, and the launch uses min(number of SMs, 160) CTAs.  A request beyond that is refused with PCAL_ERR_LIMIT;
 * nothing is launched.  There is no limit on n_samples (long segments are served in several launches).
 *
 * Sharing: EVERY call on a device uses the same array.  Calls issued to one stream are safe back to back (a call's
 * kernels start writing only after the previous call's kernels have finished), and the array needs no clearing: every
 * word a call reads it has written before (the contents left by the last call are never read).  Calls that can
 * OVERLAP on the GPU -- different streams without an event between them, different host threads on different
 * streams -- RACE on it and give wrong bins; serialise them.
 *
 * The call performs no cudaMalloc, cudaFree, cudaMallocHost or any other allocating routine, and does not synchronise.
 * The first call on each device additionally looks up the array's device address (cudaGetSymbolAddress), the number
 * of SMs and sets the kernels' shared-memory attribute: make that call once outside a graph capture.
 */
#ifndef PCAL_NOALLOC_H_
#define PCAL_NOALLOC_H_

#include "pcal.h"

#ifdef __cplusplus
extern "C" {
#endif

#define PCAL_NOALLOC_MAX_BINS 1024u
#define PCAL_NOALLOC_MAX_CTAS 160u
#define PCAL_NOALLOC_SCRATCH_BYTES (PCAL_NOALLOC_MAX_CTAS * PCAL_NOALLOC_MAX_BINS * 16u)

/*
 * P[b] (+)= sum_{n = start_index .. start_index + n_samples - 1, n = b (mod N_bins)} x[n] exp(-j 2 pi ((n F_off) mod F_s) / F_s)
 * (eq. 2.3 then eq. 2.2; frequencies snapped to the 1 micro-hertz grid as in pcal_create, reading R16).
 *
 * dev_samples   [device] packed samples of ONE channel, 16-byte aligned, caller-owned, valid until the stream work is done
 * n_samples     samples in the segment; n_samples * bits must be a multiple of 8 (else PCAL_ERR_ALIGNMENT); 0: a no-op
 *               when accumulate != 0, else the bins are set to zero
 * start_index   absolute index n of the first sample (phase origin n = 0 and bin index n mod N_bins): a stream can be
 *               cut anywhere, each segment passed with its own start index and accumulate = 1
 * f_s_hz, f_comb_hz, f_offset_hz, bits, encoding   as in pcal_create (2-bit both encodings, int8, float32)
 * accumulate    0: the bins are overwritten; else the segment's sums are added to what dev_out_bins holds
 * dev_out_bins  [device] N_bins x (re, im) doubles, 16-byte aligned, caller-owned
 * cuda_stream   the stream the work is enqueued on (asynchronous)
 *
 * Errors: PCAL_ERR_INVALID (NULL, bad frequencies / bits / encoding), PCAL_ERR_ALIGNMENT, PCAL_ERR_LIMIT (N_bins above
 * PCAL_NOALLOC_MAX_BINS), PCAL_ERR_UNSUPPORTED (lcm(N_bins, samples per load) > 256 loads: the kernel's CTA iteration
 * cannot hold a whole number of periods; samples per load = 4 for float32, 16 otherwise), PCAL_ERR_DEVICE.
 */
int pcal_fold_noalloc(const void *dev_samples, uint64_t n_samples, uint64_t start_index, double f_s_hz, double f_comb_hz,
                      double f_offset_hz, int bits, int encoding, int accumulate, double *dev_out_bins, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PCAL_NOALLOC_H_ */
