// Internal declarations shared by the host API (lloid_api.cu) and the kernels.  Not part of the ABI.
//
// Coordinates.  lloid_filter walks the caller's buffer in super-chunks [k_s, k_s + n_s)
// (A1 resamples a whole super-chunk in one launch) and each super-chunk in chunks [k_a, k_a + c),
// k_a = k_s + o.  For every detector a work strain buffer xw[H + n_s] holds the last H samples of
// history followed by the super-chunk; xw[i] is absolute sample k_s - H + i.  A rate-d stream is
// indexed from the same origin: xs_d[jj] is the decimated sample at absolute time k_s - H + d*jj, so
// a chunk's slice data starts o/d further in.  kappa = k - k_a is the chunk-local output index,
// 0 <= kappa < c; the Y rows below are chunk-local.
//   slice with d == 1 :  Y row r  <->  kappa = r                      rows [0, c)
//   slice with d  > 1 :  Y row r  <->  low-rate index floor(kappa/d) = r - K_up   rows [0, c/d + 2 K_up)
// so that for every slice   c^s[kappa] = sum_{i=-K_up}^{K_up-1} w_phi[i] rho^s[row floor(kappa/d) + K_up - i],
// phi = kappa mod d, w_phi[i] = d lp_{d,K_up}[d i + phi]   (A4 in include/lloid.h).
#pragma once
#include "../../include/lloid.h"
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>

namespace lloid {

constexpr int kKUp = 8;            // interpolation half-width supported by the kernels
constexpr int kTimeTile = 128;     // f0 samples per epilogue tile; chunk starts are aligned to it
constexpr int kMaxRates = 6;       // d in {1,2,4,8,16,32}
constexpr int kRowPad = 128;       // reconstruction rows padded to a multiple of this (fp32 path)
constexpr int kRowPad16 = 256;     // fp16 path: a CTA pair reconstructs 2 x 128 rows = 128 templates
constexpr int kMaxGroupSlices = 8; // slices of one (bin, detector) that share a rate
constexpr int kMaxF0Slices = 4;    // full-rate (d == 1) slices of one (bin, detector)
constexpr int kLPad = 32;          // basis count padded to a multiple of this

struct SliceParams {               // one per (bin, detector, slice); lives in a device table
  const float*  U32;               // [L_pad][n_taps]            fp32 path
  const float*  R32;               // [rows_pad][L_pad]          fp32 path
  const __half* U16;               // fp16 path: packed [tap block 64][tap group 8][l L_pad][8 taps] (bulk-copy source)
  const __half* U16b;              // folded slice: the odd phase's filters (U16 = even phase)
  const __half* R16;               // fp16 path: packed R16 layout (below)
  void*    Y;                      // chunk-local y^s: fp32 row-major [y_rows_cap][L_pad], or fp16 packed Y16 (below)
  int32_t  d, log2d, rate_idx;
  int32_t  n_taps, L, L_pad;
  int32_t  rows, rows_pad;         // 2N and its padding
  int32_t  jjY0;                   // xs index of Y row 0 at o = 0: (H-Delta)/d - K_up (d>1) or H-Delta (d==1)
  int32_t  y_rows_cap;             // allocated Y rows
  int32_t  bin, det, slice;
  int32_t  fir_halo;               // FIR view: rows computed per chunk = (c >> log2d) + fir_halo   (2 K_up for d > 1, else 0)
  int32_t  out_mul, out_add;       // FIR view: FIR row m is written to Y row out_mul m + out_add   (1, 0 except below)
  int32_t  y_step64;               // fp16: bytes from one 64-row tile of this slice's Y16 to the next (the record of its rate group)
  int32_t  pad_;
};
// fp16 path, "interpolation folded into the basis filters": a slice at f0 / 2 is NOT reconstructed at
// its own rate and interpolated afterwards (A3 then A4); since both steps are linear,
//   c^s_i[k] = sum_l R^s[i, l] yhat_l[k],   yhat_l[2 m + phi] = sum_u Uhat_phi[l, u] x^s[j0 + m + u],
//   Uhat_phi[l, u] = sum_i w_phi[i] U^s[l, u - K_up + i]      (n_s + 2 K_up taps, phi = 0, 1),
// i.e. TWO basis-FIR problems at the low rate write the even / odd rows of a full-rate y, and the f0 kernel reconstructs
// the slice like a d = 1 slice.  The reconstruction tables then hold the slice with d = 1; the FIR problem table
// (fir_sp) holds the two phase problems.  This halves the rho^(d) bytes that cross HBM between the two kernels.
constexpr int kFoldMaxD = 2;

struct RateParams {                // one per distinct decimation factor
  const float* taps;               // [2 K_dn d + 1], taps[u] = sqrt(d) lp[K_dn d - u]   (d == 1: unused)
  float*   xs32;                   // [D][xs_len]  (d == 1: aliases the work strain buffer)
  __half*  xs16;                   // [D][xs_len]  fp16 path only
  int32_t  d, xs_len;
  int32_t  jj_lo_fixed;            // first index needed at a chunk start: constant per bank
  int32_t  jj_hi_off;              // needed end = jj_hi_off + c/d  (exclusive)
};

struct BinParams {                 // one per (bin, detector)
  int32_t n_templates, n_slices, first_slice /* index into SliceParams table */, rows_pad;
};

struct Peak {                      // 16 bytes: per-tile partial maximum of |rho|^2 for one template
  float q; int32_t kappa; float re, im;
};

struct PeakState {                 // running in-window maximum carried across tiles, chunks and calls
  float q; float re; float im; int32_t pad; int64_t k;
};

struct Capture {                   // lloid_debug_capture
  float*  snr; int64_t k_begin, n; int32_t bd; int32_t rows;
};

// fp32 path: rho^(d) = sum over the slices of one (bin, detector) at rate d of R^s y^s, computed ONCE per chunk at the
// low rate (the fused f0 kernel then only interpolates it), fp32 row-major [rows_pad][q_cols]
struct Q32Group {
  int32_t n_slices;                // 0: no slice at this rate
  int32_t slice[kMaxGroupSlices];  // indices into the SliceParams table
  int32_t log2d, q_cols, rows_pad;
  float*  Q;
};

// Opt-in dynamic shared memory of a kernel: the architecture maximum (227 KB per CTA) minus the kernel's static part.
// A per-device, per-function attribute: set at finalize on the bank's device, always to the maximum, so banks of
// different sizes or on different devices never lower each other's limit.
template <class F> inline cudaError_t set_max_dyn_smem(F f)
{
  cudaFuncAttributes at;
  cudaError_t e = cudaFuncGetAttributes(&at, f);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - (int)at.sharedSizeBytes);
}

// ---- launchers (one translation unit per kernel family) ---------------------------------------
int configure_common_kernels();    // opt-in shared memory of every kernel of the TU, on the current device (finalize)
int configure_f32_kernels();
void launch_resample(const RateParams* rates_dev, const RateParams* rates_host, int n_rates,
                     const float* xw, int xw_pitch, int xw_valid, int n_det, int k_dn, int c,
                     bool want_f16, cudaStream_t st, int64_t* launches);

// o: offset (f0 samples) of the chunk inside the resampled super-chunk; c: chunk length
void launch_fir_f32(const SliceParams* sp_dev, const SliceParams* sp_host, int n_problems,
                    const RateParams* rates_dev, int n_det, int o, int c, cudaStream_t st, int64_t* launches);

// packed16: Y and R are the packed fp16 arrays Y16 / R16 of the tcgen05 path (fallback for banks the
// tensor reconstruction kernels do not cover)
void launch_recon_f32(const SliceParams* sp_dev, const BinParams* bp_dev, const BinParams* bp_host,
                      int n_bd, int max_rows_pad, const float* const* upw_dev, Peak* partials,
                      int tiles_cap, int max_templates, int c, int64_t k_a, Capture cap, bool packed16,
                      cudaStream_t st, int64_t* launches);

// A5/A6: one thread per (bin, detector, template, peak window touched by the chunk); state double-buffered
// fp32 path, two kernels: low-rate reconstruction GEMM, then d = 1 reconstruction + interpolation + peaks
void launch_lowrate_gemm_f32(const SliceParams* sp_dev, const Q32Group* groups_dev, const Q32Group* groups_host, int n_groups,
                             int max_rows_pad, int c, bool packed16, cudaStream_t st, int64_t* launches);
void launch_recon_f32_q(const SliceParams* sp_dev, const BinParams* bp_dev, int n_bd, int max_rows_pad,
                        const float* const* upw_dev, const Q32Group* groups_dev, Peak* partials, int tiles_cap,
                        int max_templates, int c, int64_t k_a, Capture cap, bool packed16, cudaStream_t st, int64_t* launches);

// partials: [bd][slot][template]; slot_tiles_dev[bd] = tiles per slot of that (bin, detector) (null: 1 everywhere)
void launch_merge_windows(const BinParams* bp_dev, int n_bd, int max_templates, const Peak* partials,
                          int slots_cap, const int32_t* slot_tiles_dev, int c, int64_t k_a /* host copy: launch geometry */,
                          const long long* k_base_dev /* first sample of the call, device */, int64_t k_off /* chunk - call start */,
                          int W, float theta,
                          const PeakState* state_in, PeakState* state_out, int n_det, int bin_base /* added to the bin index of every trigger */,
                          void* triggers, int64_t capacity, unsigned long long* count, cudaStream_t st, int64_t* launches);
void launch_advance_counter(long long* k_base_dev, int64_t n, cudaStream_t st);
// NEXT-2 coincidence (kernels_coinc.cu): table = int[total templates][n_det][n_w], filled with -1, then trigger indices
void launch_coincidence(const lloid_trigger_t* trig, long long n, const long long* tmpl_off_dev, int n_bins, int n_det, long long k_w0, int W,
                        int n_w, int* table, size_t table_bytes, const int* max_dt_dev, lloid_coinc_t* out, long long capacity,
                        unsigned long long* count, cudaStream_t st);

void launch_reset_state(PeakState* state, int64_t n, cudaStream_t st);

// fp16 / tcgen05 path (kernels_f16.cu: basis FIR; kernels_f16_recon.cu: reconstruction + upsample + peaks)
//
// Packed fp16 layouts (all are the tcgen05 no-swizzle K-major canonical layout: a core matrix is 8 rows x
// 8 fp16 = 128 contiguous bytes, so every operand tile is fetched with plain 1-D bulk copies):
//   Y16  [time tile of 64 rows][l / 8][row % 64][l % 8]             y^s, written by the FIR kernel; a CTA of a pair
//                                                                   supplies one 64-row tile of a 128-sample MMA tile
//   R16  [rb = i / 128][l / 8][lane(i % 128)][l % 8]                R^s; inside a 128-row block (64 templates) row
//        i = 2 p + part sits in lane 16 (p / 8) + 8 part + p % 8 (r16_lane): cosine and sine row of a template are 8
//        lanes apart, which is what one thread of a 16x256b TMEM load holds (f0 epilogue, no shuffles)
//   Q16  [rb][j / 8][lane][j % 8]                                   rho^(d) = sum over the slices at rate d of R^s y^s
//        (rows in the SAME lane order: the low-rate kernel's accumulator lanes are the f0 kernel's A-operand rows)
constexpr int kTplBlock = 128;     // complex templates per CTA PAIR (M = 256 rows: 128 per CTA)
constexpr int kNLowRates = kMaxRates - 1;
__host__ __device__ inline int r16_lane(int i_in_block) { const int p = i_in_block >> 1; return 16 * (p >> 3) + 8 * (i_in_block & 1) + (p & 7); }

struct RateGroup {                 // one per (bin, detector, distinct rate with d > 1)
  int32_t  n_slices;               // 0: this (bin, detector) has no slice at this rate
  int32_t  slice[kMaxGroupSlices]; // indices into the SliceParams table
  int32_t  log2d, q_groups_cap;    // q_groups_cap: allocated groups of 8 low-rate samples per template block
  int32_t  l_sum, n_rb;            // sum of L_pad over the group's slices; pair blocks of 128 templates
  __half*  Q;                      // [2 n_rb row blocks][q_groups_cap][128][8]
};

struct BdPlan {                    // one per (bin, detector): what the f0-rate kernel needs
  int32_t  n_f0;                   // d == 1 slices
  int32_t  f0_slice[kMaxF0Slices];
  int32_t  l_sum;                  // sum of L_pad over the d == 1 slices
  int32_t  n_templates, n_rb;
};

struct F0Combo { int32_t bd, rb; };   // (bin*detector, template block) handled back to back along time

// A4 on the tensor cores (f0_pair_kernel): one interpolation MMA = one 16-row chunk of a rate's rho^(d) window times the
// block of the band matrix P_d its rows touch.  The issuing thread reads everything an MMA needs from ONE table entry in
// the kernel parameters (uniform loads straight into uniform registers): the table is indexed by the rate, the
// alignment variant of the window and the ring slot of the window's first chunk, so the ring wrap is folded in.
struct PairMma {
  uint32_t a_off;                  // A descriptor offset (16-byte units) of the chunk's ring slot, relative to the rate's buffer
  uint32_t p_lo;                   // B descriptor low word of the block relative to the P blob: offset >> 4 | (N / 2) << 16
  uint32_t idesc;                  // cta_group::2 instruction descriptor, M = 256, N = columns of the block
  uint32_t d_col;                  // first accumulator column
};
constexpr int kPairTabMax = 224;   // table entries in the kernel parameters (3.5 KB)
struct PairRate {                  // one per distinct rate with d > 1 (bank-wide)
  int32_t  log2d;
  int32_t  adv;                    // low-rate rows per 128-sample tile: 128 / d
  int32_t  cap_chunks;             // capacity of the rate's circular buffer, in chunks of 16 rows (4 KB per CTA)
  int32_t  n_var;                  // window start is adv t: 16 / adv alignments of it inside a chunk (1 when adv >= 16)
  int32_t  ring_off;               // byte offset of the circular buffer in the window area
  int32_t  n_items[4];             // MMAs per tile, per variant
  int32_t  tab_off[4];             // per variant: table entries [slot of the first chunk][item]
};

// Static schedules of the persistent reconstruction kernels (A7): F0Sched and LowSched in kernels_f16_recon.cu.  Work =
// cells x time tiles; a cell is one stationary operand set ((bin, detector), template block -- per rate in the low-rate
// kernel); cluster i of G takes the cost range [T i / G, T (i + 1) / G) of the flattened sequence, so every SM pair
// gets the same tensor work whatever the bank geometry.
struct SchedBd {                   // one tensor-path (bin, detector) (f0 kernel) / one of its rate groups (low-rate kernel)
  int32_t bd, n_pb, w, pad;        // index (low-rate kernel: first unit), template blocks of 128, cost per tile (MMAs)
  long long cum;                   // sum of n_pb * w over the earlier entries
};

struct F16Plan;                    // opaque host-side plan: work lists, band matrices, Q buffers
F16Plan* f16_plan_create(const SliceParams* sp_host, int n_problems /* reconstruction view */,
                         const SliceParams* fir_host, int n_fir /* FIR problems */, const BinParams* bp_host, int n_bd,
                         int n_det, int chunk_cap, const double* const* up_w /* [kMaxRates]: w[(i+K_up) d + phi] or null */,
                         void* (*q_alloc)(void*, size_t) /* rho^(d) buffers: zeroed device memory or null; nullptr = cudaMalloc */, void* q_ctx,
                         int64_t* bytes, char* err, int errlen);
void f16_plan_destroy(F16Plan*);
bool f16_plan_r_tmem(const F16Plan*);          // reconstruction kernels keep the stationary R in TMEM (K <= 512)
bool f16_plan_tensor_recon(const F16Plan*);   // false: bank outside the tensor reconstruction kernels' limits
void f16_plan_disable_tensor_recon(F16Plan*);
const uint8_t* f16_plan_excluded(const F16Plan*);   // tensor_recon only: per (bin, detector) flags of the bins left to the FFMA kernels, or null
int  launch_fir_f16(F16Plan*, const SliceParams* sp_dev, const SliceParams* sp_host, int n_problems,
                    const RateParams* rates_dev, int o, int c, cudaStream_t st, int64_t* launches);
// partials of the tensor path: ONE record per (bin, detector, template, granule); a granule is a run of gt tiles
// aligned to absolute multiples of gt tiles, gt = f16_granule_tiles(W) dividing the peak window
int  f16_granule_tiles(int peak_window);
int  f16_read_trace(long long* out /* [2][8][8] */, int reset);
int  launch_recon_f16(F16Plan*, const SliceParams* sp_dev, Peak* partials, int slots_cap, int max_templates,
                      int c, int64_t k_a, int gt, float theta /* snr threshold: the epilogue's gate */, Capture cap, cudaStream_t st, int64_t* launches,
                      cudaEvent_t after_lowrate /* recorded between the two kernels when non-null */);

}  // namespace lloid
