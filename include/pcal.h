/*
 * pcal.h -- C ABI of libpcal: B200 (sm_100a) multi-tone phase-calibration (PCal) extraction.
 *
 * Method: Wagner & Pogrebenko, "Fast Multi-tone Phase Calibration Signal Extraction"
 * (cited as PAPER.md:<line> = /root/reference/PAPER.md).  The hot path is
 *     packed baseband samples --(decode)--> x[n]
 *     x^[n] = x[n] exp(-j w_offset n)            (rotation, eq. 2.3)
 *     P[b]  = sum_{n = b mod N_bins} x^[n]       (fold,     eq. 2.2)
 *     T[i]  = sum_b P[b] exp(-j 2 pi i b/N_bins) ("DFT(P)")
 * with N_bins = f_s / f_comb.  The rotator comes either from a precomputed look-up table of
 * length L = lcm(N_bins, N_rotator), N_rotator = f_s / gcd(f_s, f_offset) (eq. 2.4)
 * or from a sinewave generator with constant phase increment (eq. 2.5-2.9) whose
 * phasor is re-derived from exactly reduced integer phases at least every 2^16 samples (R14).
 *
 * Conventions: rotator sign exp(-j...) as eq. 2.3; forward unnormalised
 * DFT; sample index n = 0 at the first sample after create/reset and running across
 * pcal_extract calls; frequencies are snapped to a 1 micro-hertz integer grid and the snapped
 * values define the problem.
 *
 * All functions return PCAL_OK (0) or a negative PCAL_ERR_*; nothing throws across the ABI.
 * There is no CPU fallback: without a usable CUDA device pcal_create fails with PCAL_ERR_DEVICE.
 * Pointers are marked [host] or [device].  A context is not thread-safe; all calls on one
 * context must be issued from one thread at a time and use one CUDA stream (or be ordered
 * externally).
 */
#ifndef PCAL_H_
#define PCAL_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pcal_ctx pcal_ctx;

enum {
    PCAL_OK = 0,
    PCAL_ERR_INVALID = -1,     /* bad argument (NULL, non-integer f_s/f_comb, bad bits/encoding/channels) */
    PCAL_ERR_ALIGNMENT = -2,   /* pointer not 16-byte aligned or segment not a whole number of bytes/words */
    PCAL_ERR_STATE = -3,       /* call not legal in the current state */
    PCAL_ERR_UNSUPPORTED = -4, /* valid request this build cannot serve (e.g. LUT of impractical length) */
    PCAL_ERR_DEVICE = -5,      /* CUDA error / no device */
    PCAL_ERR_NOMEM = -6,
    PCAL_ERR_LIMIT = -7        /* size beyond the fixed scratch of the no-allocation entry point (pcal_noalloc.h) */
};

/* Sample encodings (PAPER.md:31 says only "2-bit or higher"; tables defined here, R15).
 * 2-bit OFFSET_BINARY: code c -> level 2c-3        (0:-3, 1:-1, 2:+1, 3:+3)
 * 2-bit SIGN_MAG:      code (s<<1)|m, s=1 negative, m=1 magnitude 3   (0:+1, 1:+3, 2:-1, 3:-3)
 * 8-bit TWOS_COMPLEMENT: int8 value.     32-bit IEEE_FLOAT: float32 value.
 * Packing: 2-bit single channel, 4 samples per byte, sample m in bits 2(m&3)..2(m&3)+1 of byte
 * m>>2.  2-bit with C > 1 channels (C a power of two, 2C <= 32): one field of 2C bits per time
 * sample, fields packed LSB-first into little-endian 32-bit words; channel c in bits 2c..2c+1 of
 * its field (C = 16: one uint32 per time sample). */
enum { PCAL_ENC_OFFSET_BINARY = 0, PCAL_ENC_SIGN_MAG = 1, PCAL_ENC_TWOS_COMPLEMENT = 2, PCAL_ENC_IEEE_FLOAT = 3 };

/* Rotator source for eq. 2.3. */
enum { PCAL_ROT_AUTO = 0, PCAL_ROT_LUT = 1, PCAL_ROT_GENERATOR = 2 };

#define PCAL_MAX_CHANNELS 16

typedef struct pcal_info_t {
    int32_t n_channels;
    int32_t n_bins;                 /* N_bins = f_s / f_comb */
    int32_t bits;
    int32_t encoding;
    int32_t rotator_requested;      /* PCAL_ROT_* as set */
    int32_t rotator_in_effect;      /* PCAL_ROT_LUT or PCAL_ROT_GENERATOR (LUT also when all offsets are 0) */
    int32_t integer_exact;          /* 1 if integer input and every f_offset == 0 (int64 bins valid) */
    int32_t k_shift;                /* PAPER.md:97 bin shift in effect */
    uint64_t n_processed;           /* samples per channel since create/reset */
    uint64_t fold_period;           /* M: accumulation period of the fold kernel in time samples (LUT mode) */
    uint64_t lut_len[PCAL_MAX_CHANNELS]; /* L_c = lcm(N_bins, N_rotator) per channel */
    uint64_t kernel_launches;       /* CUDA kernels launched by this context so far */
} pcal_info_t;

/*
 * Create a context (PAPER.md:37-57 problem statement).
 *   out            [host] receives the context; caller frees with pcal_destroy.
 *   f_s_hz         sample rate  > 0
 *   f_comb_hz      comb spacing > 0; f_s/f_comb must be an integer >= 2 (eq. 2.2 needs an integer
 *                  period), else PCAL_ERR_INVALID
 *   f_offset_hz    comb offset >= 0 and < f_s, applied to every channel (see pcal_set_channel_offsets)
 *   bits           2, 8 or 32;  encoding must match (2: OFFSET_BINARY|SIGN_MAG, 8: TWOS_COMPLEMENT,
 *                  32: IEEE_FLOAT)
 *   n_channels     1, or a power of two <= 16 with bits == 2
 * Uses the current CUDA device.  Allocates device accumulators; tables are built lazily at the
 * first pcal_extract.
 */
int pcal_create(pcal_ctx **out, double f_s_hz, double f_comb_hz, double f_offset_hz,
                int bits, int encoding, int n_channels);

/* Per-channel comb offsets (BASELINE.json config 4).  f_offset_hz: [host] n_channels doubles.
 * Legal only before the first pcal_extract after create/reset, else PCAL_ERR_STATE. */
int pcal_set_channel_offsets(pcal_ctx *ctx, const double *f_offset_hz);

/* Choose the rotator source.  AUTO = LUT when the fold period is practical, else GENERATOR.
 * LUT with an impractical period -> PCAL_ERR_UNSUPPORTED (reported by the next pcal_extract).  GENERATOR serves every
 * 2-bit layout (1..16 channels, each with its own offset) and every integer N_bins <= 4096 for 2-bit and int8 samples;
 * float32 samples: N_bins <= 1024 (else PCAL_ERR_UNSUPPORTED).  Legal only before the first pcal_extract after
 * create/reset. */
int pcal_set_rotator(pcal_ctx *ctx, int mode);

/* rotate by w_offset + k w_comb instead of w_offset (0 <= k < N_bins); outputs are
 * un-shifted back to natural tone order by pcal_finalize (bin reordering) and by
 * pcal_get_folded (which returns P as if k were 0).  Legal only before the first pcal_extract
 * after create/reset. */
int pcal_set_k_shift(pcal_ctx *ctx, int k);

/* Absolute index of the next sample (default 0 after create/reset).  Lets a time-sharded rank
 * start in the middle of the stream.  Same legality rule as above. */
int pcal_set_start_index(pcal_ctx *ctx, uint64_t n_start);

/*
 * Promise about the sample buffers (default 0).  The kernels of a context are launched with programmatic
 * dependent launch.  With ready != 0 the caller guarantees that every dev_samples buffer handed to
 * pcal_extract / pcal_extract_series / pcal_integrate is completely written BEFORE the call (e.g. by an
 * earlier, synchronised transfer; data resident in HBM) -- not produced by work that may still be running
 * on cuda_stream.  The streaming kernel of a call then reads its input while the kernels of the previous
 * call are still running (consecutive launches overlap; whatever it WRITES is ordered behind them on the
 * device).  With 0 it first waits for all earlier work of the stream, like any
 * kernel.  Results are identical either way.
 */
int pcal_set_input_ready(pcal_ctx *ctx, int ready);

/*
 * Rotate + fold one segment (eq. 2.3 + eq. 2.2) into the context's accumulators.
 *   dev_samples    [device] 16-byte aligned, caller-owned, valid until the stream work completes
 *   n_samples      samples PER CHANNEL in this segment; n_samples*bits*n_channels must be a
 *                  multiple of 8 (whole bytes), else PCAL_ERR_ALIGNMENT.  0 is a no-op.
 *   cuda_stream    cudaStream_t (NULL = default stream).  Asynchronous: never synchronises.
 * Successive calls are one continuous stream: the result is invariant to the split points.
 * All calls on one context must use one stream, or be ordered by the caller (a context is not thread-safe).
 */
int pcal_extract(pcal_ctx *ctx, const void *dev_samples, uint64_t n_samples, void *cuda_stream);

/*
 * A time series of integrations in one call ("112 integrated time-integrated PCal
 * results", 10 s each): period k = samples [k, k+1)*n_per_period of the segment.  The accumulators
 * restart at every period, the sample index (rotator phase, bin alignment) runs on, so period k equals
 * what pcal_set_start_index(n0 + k*n_per_period) + pcal_extract + pcal_finalize would give.
 *   dev_samples     [device] 16-byte aligned; n_per_period*bits*n_channels must be a multiple of 128
 *                   (every period starts 16-byte aligned), else PCAL_ERR_ALIGNMENT
 *   dev_out_tones   [device] n_periods*n_channels*N_bins*2 doubles: T of every period (layout of
 *                   pcal_finalize per period)
 *   dev_out_folded  [device] same size or NULL: P of every period (needs k_shift == 0)
 * Asynchronous on cuda_stream.  Afterwards the context holds the LAST period's accumulators.
 */
int pcal_extract_series(pcal_ctx *ctx, const void *dev_samples, uint64_t n_per_period, uint32_t n_periods,
                        void *cuda_stream, double *dev_out_tones, double *dev_out_folded);

/* Same, with the segment in [host] memory (pinned for full speed): copies it to the device in
 * chunks on cuda_stream and extracts each chunk.  Returns after the last copy has been enqueued
 * and the host buffer may be reused (it synchronises the stream). */
int pcal_extract_host(pcal_ctx *ctx, const void *host_samples, uint64_t n_samples, void *cuda_stream);

/*
 * Tone spectrum: reduce + N_bins-point DFT of the folded period, copy to the host,
 * synchronise the stream.
 *   out_tones      [host] n_channels*N_bins*2 doubles; out[(c*N_bins + i)*2 + {0,1}] = Re, Im of
 *                  T[c][i], natural tone order: tone i sits at frequency i*f_comb + f_offset,c.
 * Does not reset: integration may continue and finalize may be called again.
 */
int pcal_finalize(pcal_ctx *ctx, double *out_tones);

/* As pcal_finalize but only enqueues (DFT + async copy into out_tones, which should be pinned
 * host memory) on the context's stream; the caller synchronises.  When out_tones is device-visible
 * pinned memory the DFT kernel writes it directly; that property is looked up when the pointer changes
 * from the previous call, so a buffer must not be freed and re-created at the same address with a
 * different kind of memory between two calls. */
int pcal_finalize_async(pcal_ctx *ctx, double *out_tones);

/*
 * One integration period in one call ("single integration ... 10 seconds"; the caller's
 * loop over periods): pcal_reset, pcal_extract(dev_samples, n_samples, cuda_stream) and
 * pcal_finalize_async(out_tones), with the argument rules of those calls.  Nothing else is added; it
 * exists so that a host loop over short periods costs one library call per period.  Asynchronous.
 */
int pcal_integrate(pcal_ctx *ctx, const void *dev_samples, uint64_t n_samples, void *cuda_stream, double *out_tones);

/*
 * PCal data analysis on the device (R23-R25): enqueues the DFT and
 * one analysis kernel, copies the results to the host, synchronises the stream.
 *   out_summary    [host] n_channels*PCAL_N_SUMMARY doubles, per channel:
 *                  [0] b*      bin of the largest |P[b]|^2 (first one on ties)
 *                  [1] delta   three-point vertex offset in (-1/2, 1/2), cyclic neighbours
 *                  [2] pulse (group) delay (b* + delta)/f_s in seconds (bin i <-> delay i/f_s)
 *                  [3] |P[b*]|^2   [4] sum_b |P[b]|^2
 *                  [5] cable delay t_d of eq. 2.1 from the least-squares slope of the unwrapped tone
 *                      phases arg T[i] + pi/2 over the in-band tones (branch |t_d| < 1/(2 f_comb))
 *                  [6] intercept of that line in radians   [7] rms residual in radians
 *   out_bandpass   [host] n_channels*N_bins*2 doubles or NULL: group-delay corrected band-pass
 *                  B[c][i] = T[c][i] exp(+j 2 pi i (b* + delta)/N_bins).
 */
#define PCAL_N_SUMMARY 8
int pcal_analyze(pcal_ctx *ctx, double *out_summary, double *out_bandpass);

/*
 * Multi-pass counter-rotation ("short integration times combined with multiple passes over the
 * x[n] input data, iteratively counter-rotating the input data using the residual phase shift detected in the
 * previous pass"; reading R27).
 *
 * pcal_residual_rotation: the residual phase shift of one pass.  dev_series_tones = [device] the output of
 * pcal_extract_series ([n_periods][n_channels][N_bins] complex128).  Per channel,
 *   S = sum_{m < n_periods-1} sum_{i in band} T_{m+1}[i] conj(T_m[i]),  band = tones 0 (1 when that channel's
 *   f_offset is 0: that tone is sin(0)) .. N_bins/2 - 1,
 * and out[c*PCAL_N_RESIDUAL + {0,1,2}] = arg S (radians per period; = 2 pi (f_true - f_rot) n_per_period/f_s),
 * |S|, sum |T_{m+1}[i]| |T_m[i]| (|S| over it = coherence in [0,1]).  out: [host].  Synchronises the context's stream.
 *
 * pcal_refine_offset: the passes.  Single-channel contexts only (else PCAL_ERR_UNSUPPORTED).  Starting from the
 * context's f_offset, each pass extracts n_periods short integrations of n_per_period samples from dev_samples
 * ([device], the rules of pcal_extract_series) at the current rotator frequency, measures the residual phase
 * shift and counter-rotates: f_rot <- f_rot + arg S / (2 pi T_int), T_int = n_per_period / f_s, on the 1 micro-hertz
 * grid; stops when |arg S| <= tol_rad or after max_passes passes.  Unambiguous for |f_true - f_rot| < 1/(2 T_int).
 *   out_f_offset_hz [host] the last rotator frequency set;  out_history [host] max_passes*4 doubles or NULL: per
 *   pass (f_rot used, arg S, |S|, norm);  out_passes [host] passes run.
 * On success the context is reset and ITS f_offset is replaced by the refined value, so that the caller can go on
 * to the long coherent integration (pcal_extract + pcal_finalize / pcal_analyze).  Synchronous.
 */
#define PCAL_N_RESIDUAL 3
int pcal_residual_rotation(pcal_ctx *ctx, const double *dev_series_tones, uint32_t n_periods, double *out);
int pcal_refine_offset(pcal_ctx *ctx, const void *dev_samples, uint64_t n_per_period, uint32_t n_periods, void *cuda_stream,
                       uint32_t max_passes, double tol_rad, double *out_f_offset_hz, double *out_history, uint32_t *out_passes);

/* Folded period P before the DFT: [host] n_channels*N_bins*2 doubles (Re, Im).  Synchronises. */
int pcal_get_folded(pcal_ctx *ctx, double *out_bins);

/* Exact integer bins: [host] n_channels*N_bins int64.  Valid only for integer input with every
 * f_offset == 0 and k_shift == 0 (else PCAL_ERR_STATE).  Synchronises. */
int pcal_get_folded_i64(pcal_ctx *ctx, int64_t *out_bins);

/* Add externally obtained folded bins (same layout as pcal_get_folded) into the accumulators:
 * the exchange step of a time-sharded multi-GPU run. */
int pcal_add_folded(pcal_ctx *ctx, const double *bins);

/* Device-resident variants of pcal_get_folded / pcal_add_folded for an exchange that stays on the
 * GPU (NCCL all-gather of the bins): dev_bins is [device] n_channels*N_bins*2 doubles.  Asynchronous
 * on the context's stream.  They move the raw accumulators (no k_shift un-shifting): every rank of
 * a sharded run must use the same k_shift. */
int pcal_get_folded_dev(pcal_ctx *ctx, double *dev_bins);
int pcal_add_folded_dev(pcal_ctx *ctx, const double *dev_bins);

/* The exchange step in one launch: accumulators <- sum over r of dev_parts[r] (r = 0..n_parts-1, in that
 * order: deterministic), dev_parts = [device] n_parts contiguous blocks in the layout of pcal_get_folded_dev
 * (e.g. the output of an NCCL all-gather of every rank's bins).  Replaces the previous contents. */
int pcal_set_folded_sum_dev(pcal_ctx *ctx, const double *dev_parts, uint32_t n_parts);

/* The same for a time series of integrations with ONE exchange for all its periods: every rank folded
 * its time shard of each of n_periods periods and the bins were gathered into dev_parts = [device]
 * [n_parts][n_periods][n_channels][N_bins] complex128.  dev_out_folded [device] [n_periods][n_channels][N_bins] receives the
 * rank-order sums (P of every period), dev_out_tones [device] (same shape) their DFT (layout of pcal_finalize per
 * period).  Asynchronous on the context's stream; the context's own accumulators are not touched. */
int pcal_finalize_series_sum_dev(pcal_ctx *ctx, const double *dev_parts, uint32_t n_parts, uint32_t n_periods,
                                 double *dev_out_folded, double *dev_out_tones);

/*
 * Accuracy of the sinewave generators over many cycles (eq. 2.6/2.7, PAPER.md:142-153
 * direct method, PAPER.md:97 k-shift; R26).  One device thread per case runs the
 * recursion for n = 1..n_steps with every operation rounded once to the case's precision and records
 * out_err[case*n_chk + j] = max over the j-th of n_chk equal intervals of |y[n] - exp(-j n dphi)|, the
 * exact phasor taken from the exactly reduced integer phase (fp64).  For a k-shift give
 * f_rot_hz = f_offset + k f_comb.  cases: [host]; out_err: [host] n_cases*n_chk doubles.  Synchronous,
 * default stream of the current device, no context needed.
 */
enum { PCAL_GEN_CFO = 0, PCAL_GEN_MCO = 1, PCAL_GEN_DFR = 2, PCAL_GEN_DFR_FMA = 3, PCAL_GEN_DIRECT = 4 };
typedef struct pcal_gen_case_t {
    int32_t form;        /* PCAL_GEN_* */
    int32_t precision;   /* 32 or 64 (PCAL_GEN_DIRECT always computes its phase in float32) */
    double f_s_hz;
    double f_rot_hz;     /* rotator frequency, 0 <= f_rot < f_s */
} pcal_gen_case_t;
int pcal_generator_study(const pcal_gen_case_t *cases, uint32_t n_cases, uint64_t n_steps, uint32_t n_chk,
                         double *out_err);

/* Zero accumulators, sample index <- 0 (on the context's stream); parameters are kept. */
int pcal_reset(pcal_ctx *ctx);

/* Free everything.  NULL-safe. */
void pcal_destroy(pcal_ctx *ctx);

/* Describe the context.  info: [host]. */
int pcal_info(const pcal_ctx *ctx, pcal_info_t *info);

/* Static string for an error code. */
const char *pcal_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* PCAL_H_ */
