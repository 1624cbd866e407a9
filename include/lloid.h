/* lloid.h — C ABI of the B200-native LLOID matched-filter hot path (arXiv:2410.16416).
 *
 * What the library computes.  For every SVD bin b and detector D the LLOID filter of the paper
 * (§II.A: "downsamples the conditioned data, cross-correlates it with orthogonal
 * templates, performs matrix multiplication of the orthogonal SNR time series with SVD coefficients,
 * and finally up-samples and sums the physical SNR segments"; §II.B, multi-bank batching)
 * followed by the trigger generator ("peaks in the SNR time series with SNR > 4";
 * PAPER.md:55 triggers are formed on the device so the dense SNR never crosses to the host):
 *
 *   A1  x^s[j]     = sqrt(d_s) * sum_n lp_{d_s,K_dn}[n] x[d_s j - n]            (per detector, per rate)
 *   A2  y^s_l[j]   = sum_t U^s[l,t] x^s[j - n_s + t]                            (basis FIR, end-exclusive)
 *   A3  rho^s_i[j] = sum_l R^s[i,l] y^s_l[j]                                    (reconstruction)
 *   A4  rho_i[k]   = sum_s sum_j rho^s_i[j] d_s lp_{d_s,K_up}[k - Delta_s - d_s j]   (upsample, delay, sum)
 *   A5  per template p and window w=[wW,(w+1)W): k* = first argmax_k rho_2p[k]^2 + rho_2p+1[k]^2
 *   A6  trigger (bin, detector, p, k*, Re, Im) iff |rho|(k*) > threshold
 *
 * lp_{d,K}[n] = (1/d) sinc(n/d) (1/2)(1 + cos(pi n/(K d))), |n| <= K d, normalised to unit sum
 * (readings R1-R3).  Notation as in SURVEY.md §8.0 / DESIGN.md §1.
 *
 * Conventions.  All functions return LLOID_OK (0) or a negative lloid_status; lloid_last_error()
 * gives a thread-local, library-owned, NUL-terminated message for the last failure on this thread.
 * "host" / "device" is stated for every pointer.  The library never takes ownership of caller
 * memory.  create / upload / finalize / destroy / reset are host-synchronous and not thread-safe
 * per handle.  lloid_filter only enqueues work on the given CUDA stream: it does not allocate device memory,
 * does not synchronise the device and does not read device results on the host (the first call with a new
 * buffer length sorts one work list on the host and uploads it from pinned memory).
 * There is no CPU fallback: every entry point that needs the GPU fails with LLOID_ECUDA without one.
 */
#ifndef LLOID_H
#define LLOID_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lloid_bank lloid_bank_t;   /* opaque; created by lloid_bank_create, freed by lloid_destroy */

typedef enum {
  LLOID_F32 = 0,    /* fp32 operands, fp32 FMA accumulate (CUDA cores); 1e-3 absolute SNR parity    */
  LLOID_F16 = 1,    /* fp16 operands (x^s, U, y, R, rho^s), fp32 accumulate on tcgen05 tensor cores */
  LLOID_BF16 = 2    /* reserved; rejected with LLOID_EINVAL in this version                        */
} lloid_precision_t;

typedef enum {
  LLOID_OK = 0,
  LLOID_EINVAL = -1,     /* bad argument or inconsistent geometry                                  */
  LLOID_ENOMEM = -2,     /* host or device allocation failed                                       */
  LLOID_ECUDA = -3,      /* a CUDA runtime/driver call failed, or no sm_100 device                 */
  LLOID_ESTATE = -4,     /* upload after finalize, filter before finalize, missing slice upload    */
  LLOID_EOVERFLOW = -5   /* returned by lloid_check_count: trigger buffer was too small            */
} lloid_status;

typedef struct {
  int32_t n_bins;            /* B                                                                  */
  int32_t n_detectors;       /* D                                                                  */
  int32_t full_rate_hz;      /* f0, e.g. 2048                                                      */
  int32_t peak_window;       /* W in f0 samples (e.g. 2048); multiple of 128                       */
  float   snr_threshold;     /* theta; trigger iff |rho| > theta (strict)             */
  int32_t k_down;            /* K_dn: decimation kernel half-width in low-rate zero crossings (16) */
  int32_t k_up;              /* K_up: interpolation kernel half-width (8); must be 8 in this version */
  int32_t precision;         /* lloid_precision_t                                                  */
  int32_t device;            /* CUDA device ordinal                                                */
  int32_t max_chunk;         /* 0 = automatic; else internal time-chunk length in f0 samples
                                (multiple of 128): lloid_filter walks the buffer in chunks of this
                                size so that intermediates stay bounded / L2-resident              */
} lloid_bank_config_t;

typedef struct {             /* per bin: geometry shared by that bin's detectors                   */
  int32_t n_templates;       /* N complex templates; 2N real rows, row 2p = cos, 2p+1 = sin        */
  int32_t n_slices;          /* S                                                                  */
  int64_t template_len;      /* M in f0 samples                                                    */
} lloid_bin_desc_t;

typedef struct {             /* per (bin, slice); slice 0 is the latest part of the template       */
  int32_t rate_hz;           /* f_s; f0 / f_s must be a power of two in [1, 32]                    */
  int32_t n_taps;            /* n_s                                                                */
  int32_t n_basis;           /* L_s <= 512                                                         */
  int32_t reserved;
  int64_t end_delay;         /* Delta_s = M - b_s in f0 samples, multiple of d_s                   */
} lloid_slice_desc_t;

typedef struct {             /* 32 bytes, written by the device                                    */
  int32_t bin;
  int32_t detector;
  int32_t template_idx;      /* p in [0, N)                                                        */
  int32_t reserved;
  int64_t sample;            /* absolute f0 sample index k* since create/reset (end-exclusive: a
                                signal whose template occupies x[e-M, e) peaks at k* = e)          */
  float   snr_re;            /* rho_2p[k*]                                                         */
  float   snr_im;            /* rho_2p+1[k*];  |rho| = hypot(re, im)                               */
} lloid_trigger_t;

/* Create an empty bank.  `bins` is a host array [n_bins]; `slices` is a host array of n_bins host
 * pointers, slices[b] pointing at bins[b].n_slices descriptors.  Everything is copied.  Validates:
 * rates (power-of-two decimation <= 32), Delta_s multiple of d_s, slices tile [0, M) back to front
 * (Delta_0 = 0, Delta_{s+1} = Delta_s + d_s n_s, last slice ends at M), and causality
 * Delta_s >= (K_dn + K_up) d_s for every slice with d_s > 1.  Errors: LLOID_EINVAL, LLOID_ECUDA
 * (no such device / not compute capability 10.x), LLOID_ENOMEM. */
int lloid_bank_create(lloid_bank_t **out, const lloid_bank_config_t *cfg,
                      const lloid_bin_desc_t *bins, const lloid_slice_desc_t *const *slices);

/* Upload the SVD factors of one (bin, detector, slice) ("SVD bank"; PAPER.md:85 one bank
 * per instrument).  `basis`: host, float64, row-major [L_s][n_s], rows orthonormal (U^s).
 * `recon`: host, float64, row-major [2N][L_s] (R^s).  Both are converted to the compute precision,
 * zero-padded and re-tiled into the kernels' layout on the device; the caller keeps ownership and
 * may free them on return.  Errors: LLOID_EINVAL (indices), LLOID_ESTATE (after finalize). */
int lloid_bank_upload_slice(lloid_bank_t *bank, int32_t bin, int32_t detector, int32_t slice,
                            const double *basis, const double *recon);

/* Same arrays for several detectors of a bin at once (the paper replicates one bank):
 * identical to calling lloid_bank_upload_slice for detector = 0..n_detectors-1, but the device copy
 * is shared.  Provided so that replicated benchmark banks do not multiply device memory. */
int lloid_bank_upload_slice_shared(lloid_bank_t *bank, int32_t bin, int32_t slice,
                                   const double *basis, const double *recon);

/* Share bin `src_bin`'s device arrays with bin `dst_bin` (same geometry required, all detectors);
 * the replicated-bank construction of the paper's benchmark. */
int lloid_bank_alias_bin(lloid_bank_t *bank, int32_t dst_bin, int32_t src_bin);

/* Check that every (bin, detector, slice) was uploaded, allocate history / work buffers, build the
 * work lists.  After this call uploads are rejected and lloid_filter is allowed. */
int lloid_bank_finalize(lloid_bank_t *bank);

/* Filter the next n_samples of strain of every detector and append triggers.
 *   strain_dev      device, float32, [n_detectors][n_samples], row stride = n_samples
 *   n_samples       > 0, multiple of the largest decimation factor in the bank
 *   triggers_dev    device, lloid_trigger_t[capacity]; order within a call is unspecified
 *   n_triggers_dev  device, one int64: set to the number of triggers produced by THIS call; if it
 *                   exceeds `capacity` only the first `capacity` records were stored (overflow is
 *                   never silent: check with lloid_check_count after copying the count to the host)
 *   cuda_stream     cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default
 * The buffer is consumed as the continuation of everything fed since create/reset: strain history,
 * the running in-window peak of every template and the absolute sample counter are carried, so
 * feeding a stream in pieces gives the same triggers as feeding it at once (A8, BASELINE config 5).
 * Only windows completed by this call emit triggers.  Asynchronous; the strain buffer must stay
 * valid until the stream has finished the call.  Errors: LLOID_EINVAL, LLOID_ESTATE, LLOID_ECUDA.
 * The strain must be FINITE and is not checked: a NaN or Inf sample makes every SNR value whose filter
 * span covers it non-finite, a non-finite |rho|^2 never wins the peak comparison, so the templates of
 * that detector emit no trigger until the sample has left the carried history (H samples, about the
 * template length).  Remove such samples first (the pipeline's gating step, "conditioned
 * data": outside this path); the fp16 path additionally needs |x^s| < 65504 after the sqrt(d) gain. */
int lloid_filter(lloid_bank_t *bank, const float *strain_dev, int64_t n_samples,
                 lloid_trigger_t *triggers_dev, int64_t capacity, int64_t *n_triggers_dev,
                 void *cuda_stream);

/* CUDA graphs (low-latency streaming, BASELINE config 5).  lloid_filter only enqueues work, so a call can be captured
 * in a CUDA graph and replayed for every following buffer of the same length: the absolute sample index that triggers
 * carry is read from device memory, which every call advances on the stream.  Conditions, checked by lloid_graph_safe
 * (returns 1 / 0): n_samples and the number of samples consumed so far are multiples of peak_window (every call then
 * makes the same host-side decisions).  Protocol: make at least one eager lloid_filter call with this n_samples (the
 * first call with a new buffer length builds a work list on the host and is refused during capture); capture ONE call;
 * before every replay call lloid_graph_advance(bank, n_samples), which keeps the host-side sample counter in step.
 * The buffers captured (strain, triggers, count) are the ones every replay uses. */
int lloid_graph_safe(const lloid_bank_t *bank, int64_t n_samples);
int lloid_graph_advance(lloid_bank_t *bank, int64_t n_samples);

/* Same call with HOST buffers (the end-to-end path): `strain_host` float32 [D][n_samples] is copied
 * to a library-owned device staging buffer, filtered, and the count plus min(count, capacity)
 * triggers are copied back to `triggers_host` / `*n_triggers_host`; the call returns after the
 * stream has finished (one synchronisation).  Pinned host memory makes the copies asynchronous.
 * Returns LLOID_EOVERFLOW if count > capacity (the first `capacity` triggers are valid). */
int lloid_filter_host(lloid_bank_t *bank, const float *strain_host, int64_t n_samples,
                      lloid_trigger_t *triggers_host, int64_t capacity, int64_t *n_triggers_host,
                      void *cuda_stream);

/* LLOID_OK if count <= capacity else LLOID_EOVERFLOW (helper for callers of the async lloid_filter). */
int lloid_check_count(int64_t count, int64_t capacity);

/* Zero the strain history, the running peaks and the sample counter (enqueued on the stream). */
int lloid_reset(lloid_bank_t *bank, void *cuda_stream);

/* Test-only dense SNR capture (BASELINE asks for SNR-level parity).  Arms a capture for (bin,
 * detector): subsequent lloid_filter calls also store rho_i[k] for k in [k_begin, k_begin + n) and
 * i < 2N into snr_dev (device, float32, row-major [2N][n]) from the SAME fused kernel that finds the
 * peaks (samples outside the filtered range are left untouched).  snr_dev = NULL disarms. */
int lloid_debug_capture(lloid_bank_t *bank, int32_t bin, int32_t detector, int64_t k_begin, int64_t n,
                        float *snr_dev);

/* Introspection: absolute number of f0 samples consumed so far; internal chunk length; the number of
 * kernels launched by the last lloid_filter call; bytes of device memory held by the bank. */
int64_t lloid_samples_consumed(const lloid_bank_t *bank);
int64_t lloid_chunk_samples(const lloid_bank_t *bank);
int64_t lloid_last_launch_count(const lloid_bank_t *bank);
int64_t lloid_device_bytes(const lloid_bank_t *bank);

/* Which kernels a finalized bank runs on (introspection for tests and benchmarks): out[0] = 1 if the fp16 bank's
 * reconstruction runs on the tcgen05 kernels, out[1] = 1 if those keep the stationary reconstruction matrix in TMEM
 * (banks whose full-rate slices have more basis filters than fit shared memory), out[2] = number of (bin, detector)
 * pairs left to the CUDA-core reconstruction kernels, out[3] = number of (bin, slice) pairs whose interpolation is
 * folded into the basis filters.  All zero for an fp32 bank.  out: host, int32[4]. */
int lloid_path_info(const lloid_bank_t *bank, int32_t *out);

/* Time (ms, CUDA events on the call's stream) spent by the last lloid_filter call in each stage:
 * out_ms[0..5] = resample, basis FIR, reconstruction+epilogue (both kernels of the fp16 path), peak
 * merge/compaction, whole call, and the low-rate reconstruction kernel's share of [2] (fp16 path; else 0).
 * Only recorded when enabled with lloid_set_profiling(bank, 1) (which makes lloid_filter record
 * events; reading them synchronises on the last event).  Used by bench.py for the roofline leg. */
int lloid_set_profiling(lloid_bank_t *bank, int32_t enable);
int lloid_last_stage_ms(lloid_bank_t *bank, float *out_ms /* host, float[6] */);

/* ---- coincidence (the step after the trigger generator) --------------------------------------
 * "These triggers are passed to the coincidence generator, which identifies coincidences between triggers
 * detected with the same template and within the light travel time between detectors."  Two triggers of ONE lloid_filter
 * pass are coincident iff they have the same bin and template, different detectors a < b, and |sample_a - sample_b| <=
 * max_dt[a * n_detectors + b] (the light travel time between a and b plus the timing resolution, in f0 samples; the caller
 * chooses it: e.g. 21 + 10 samples at 2048 Hz for a 10 ms baseline).
 *   triggers_dev   device, the records of one pass over absolute samples [k_begin, k_begin + n_samples): at most one per
 *                  (bin, detector, template, peak window), which is what lloid_filter emits; records outside that range or
 *                  with indices outside the bank are ignored; of two records with the same key one is ignored
 *   n_triggers     host value, number of records (min(count, capacity) of the filter call)
 *   max_dt         host, int32 [n_detectors][n_detectors], only a < b is read; 0 <= max_dt <= peak_window
 *   scratch_dev    device, lloid_coincidence_scratch_bytes(bank, k_begin, n_samples) bytes, owned by the caller, overwritten
 *   pairs_dev      device, lloid_coinc_t[capacity]: indices into triggers_dev, a = the lower-numbered detector's trigger;
 *                  order unspecified.  n_pairs_dev: device int64, number of coincident pairs found; beyond capacity they
 *                  are counted, not stored (lloid_check_count)
 * A trigger can belong to several pairs (three detectors: ab, ac, bc are reported separately).  Asynchronous on cuda_stream;
 * no device allocation.  Errors: LLOID_EINVAL, LLOID_ESTATE (bank not finalized), LLOID_ECUDA. */
typedef struct { int64_t a, b; } lloid_coinc_t;
int64_t lloid_coincidence_scratch_bytes(const lloid_bank_t *bank, int64_t k_begin, int64_t n_samples);
int lloid_coincidence(const lloid_bank_t *bank, const lloid_trigger_t *triggers_dev, int64_t n_triggers, int64_t k_begin,
                      int64_t n_samples, const int32_t *max_dt, void *scratch_dev, int64_t scratch_bytes,
                      lloid_coinc_t *pairs_dev, int64_t capacity, int64_t *n_pairs_dev, void *cuda_stream);

/* ---- allocation-free entry point -----------------------------------------------------------------------------------
 * Steps A5 + A6 alone ("identifies peaks in the SNR time series with SNR > 4 ... 'triggers'") on a dense SNR
 * series the caller already holds in device memory, for callers that may not allocate (CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc).  Needs no bank.  It calls no cudaMalloc / cudaFree / allocating routine: its scratch
 * -- one 16-byte partial peak per template and 128-sample tile -- is a file-scope device array of
 * lloid_noalloc_max_records() = 524288 records (8 MiB), which every GPU that loads the library holds until exit.
 *   snr_dev          device, float32 [2 n_templates][row_stride], 16-byte aligned: row 2p = Re rho_p, row 2p+1 = Im rho_p;
 *                    column j is absolute sample k_begin + j
 *   n_templates      1 ... 65536;  n_templates * (n_samples / 128) <= lloid_noalloc_max_records(), else LLOID_EINVAL
 *                    (the message says so: split the call in time at window boundaries, or over templates)
 *   n_samples        positive multiple of 128;  row_stride >= n_samples, multiple of 4;  k_begin >= 0, multiple of 128
 *   peak_window      W, multiple of 128: windows [wW, (w+1)W) of ABSOLUTE sample indices; only windows that lie completely
 *                    inside [k_begin, k_begin + n_samples) emit
 *   snr_threshold    theta: trigger iff |rho|(k*) > theta (strict), k* the first maximum of |rho|^2 in the window
 *   bin, detector    copied into the records
 *   triggers_dev     device, lloid_trigger_t[capacity], order unspecified;  n_triggers_dev: device int64, set to the number
 *                    of triggers found (cleared on the stream first); beyond `capacity` records are counted, not stored
 * Asynchronous on cuda_stream, uses the CURRENT device.  The first call on a device looks the array's address up
 * (cudaGetSymbolAddress; lloid_noalloc_setup() does only that, e.g. before a capture begins).  All calls on a device share
 * the array, which keeps the last call's contents (nothing in it needs clearing: every record read is written by the same
 * call first).  Calls that OVERLAP on the GPU race on it: keep them on one stream or order them with events.
 * Errors: LLOID_EINVAL, LLOID_ECUDA. */
int64_t lloid_noalloc_max_records(void);
int lloid_noalloc_setup(void);
int lloid_window_peaks_noalloc(const float *snr_dev, int32_t n_templates, int64_t n_samples, int64_t row_stride,
                               int64_t k_begin, int32_t peak_window, float snr_threshold, int32_t bin, int32_t detector,
                               lloid_trigger_t *triggers_dev, int64_t capacity, int64_t *n_triggers_dev,
                               void *cuda_stream);

void lloid_destroy(lloid_bank_t *bank);
const char *lloid_last_error(void);
const char *lloid_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LLOID_H */
