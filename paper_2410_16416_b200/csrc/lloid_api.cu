// Host side of the C ABI in include/lloid.h: bank construction, packing, the chunk scheduler that
// drives the kernels, history carry (A8), profiling hooks.  No torch types, no CPU fallback.
#include "../../include/lloid.h"
#include "lloid_internal.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <string>
#include <vector>

using namespace lloid;

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...)
{
  char buf[512];
  va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
  g_err = buf;
  return code;
}

}  // namespace

// other translation units of the library (kernels_noalloc.cu) report through the same thread-local message
namespace lloid { void set_last_error(const char* msg) { g_err = msg ? msg : ""; } }

namespace {

#define CU(call)                                                                              \
  do { cudaError_t e_ = (call);                                                               \
       if (e_ != cudaSuccess) return fail(LLOID_ECUDA, "%s failed: %s (%s:%d)", #call,        \
                                          cudaGetErrorString(e_), __FILE__, __LINE__); } while (0)

inline int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
inline int64_t round_up(int64_t v, int64_t m) { return (v + m - 1) / m * m; }

// lp_{d,K}[n], n = -K d..K d (index n + K d): Hann-windowed sinc, unit DC gain (include/lloid.h; DESIGN R1).
// Written independently of oracle/ (no shared code): double precision, evaluated once at finalize.
std::vector<double> lowpass(int d, int K)
{
  const int half = K * d;
  std::vector<double> lp(2 * half + 1);
  const double pi = 3.14159265358979323846;
  double sum = 0.0;
  for (int n = -half; n <= half; ++n) {
    const double x = (double)n / d;
    const double sinc = (n == 0) ? 1.0 : std::sin(pi * x) / (pi * x);
    const double v = (1.0 / d) * sinc * 0.5 * (1.0 + std::cos(pi * n / (double)half));
    lp[n + half] = v; sum += v;
  }
  for (double& v : lp) v /= sum;
  return lp;
}

struct SliceHost {
  int rate, d, log2d, n_taps, L, L_pad; int64_t end_delay;
  bool fold;                       // fp16: interpolation folded into the basis filters
  // fp16: the packed basis filters are stored in COLUMN BLOCKS of at most 160 filters, each a basis-FIR problem of its own.
  // The FIR kernel keeps 512 / L_pad time tiles of accumulators in TMEM and streams all of U once per such group of tiles:
  // at L_pad = 320 that is one tile per 2 MB of U (L2-bandwidth-bound on config 4); two blocks of 160 run three tiles each.
  int n_ub = 1, ub_w[4] = {0, 0, 0, 0}, ub_l0[4] = {0, 0, 0, 0};
  void set_blocks(bool f16)
  {
    n_ub = 1; ub_w[0] = L_pad; ub_l0[0] = 0;
    if (!f16 || L_pad < 224 || getenv("LLOID_NO_USPLIT")) return;
    n_ub = std::max(2, (L_pad + 159) / 160);
    const int w = ((L_pad + n_ub - 1) / n_ub + 31) / 32 * 32;
    for (int i = 0, l0 = 0; i < n_ub; ++i, l0 += w) { ub_l0[i] = l0; ub_w[i] = std::min(w, L_pad - l0); }
  }
  size_t ub_off(int i, int n_kb) const { return (size_t)n_kb * 64 * ub_l0[i]; }    // halves before block i in a packed array
};
struct BinHost { int N, S, rows_pad; int64_t M; std::vector<SliceHost> slices; };

}  // namespace

struct lloid_bank {
  lloid_bank_config_t cfg{};
  std::vector<BinHost> bins;
  bool finalized = false;
  bool f16 = false;
  int n_bd = 0, max_templates = 0, max_rows_pad = 0, d_max = 1;
  std::vector<SliceParams> sp_host;      // reconstruction view: one per (bin, detector, slice); a folded slice has d = 1 here
  std::vector<SliceParams> fir_host;     // fp16 path: basis-FIR problems (a folded slice contributes one per output phase)
  SliceParams* fir_dev = nullptr;
  std::vector<BinParams> bp_host;
  std::vector<uint8_t> uploaded;
  std::vector<RateParams> rates_host;
  SliceParams* sp_dev = nullptr;
  BinParams* bp_dev = nullptr;
  RateParams* rates_dev = nullptr;
  float* xw = nullptr;
  float* hist = nullptr;
  int H = 0, C = 0, xw_pitch = 0, tiles_cap = 0;
  int slots_cap = 0, gt = 1;             // partial peaks: slots per chunk and (tensor path) tiles per granule
  int32_t* slot_tiles_dev = nullptr;     // [n_bd] tiles per partial slot (null: 1 everywhere)
  int S = 0;                             // super-chunk: samples resampled by one A1 launch (multiple of C)
  PeakState* state = nullptr;            // [2][n_bd][max_templates], double-buffered per chunk
  int state_cur = 0;
  Peak* partials = nullptr;
  const float** upw_dev = nullptr;
  std::vector<void*> owned;
  int64_t consumed = 0, bytes = 0, last_launches = 0;
  int64_t call_start = 0;                // absolute index of the current call's first sample (host copy)
  long long* k_base_dev = nullptr;       // the same on the device: read by the merge kernel, advanced at the end of every call
  Capture cap{nullptr, 0, 0, -1, 0};
  float* stage_strain = nullptr; size_t stage_strain_elems = 0;
  lloid_trigger_t* stage_trig = nullptr; int64_t stage_trig_cap = 0;
  unsigned long long* stage_count = nullptr;
  bool prof = false;
  std::vector<cudaEvent_t> events; std::vector<int> event_tag; size_t events_used = 0;
  F16Plan* plan16 = nullptr;
  std::vector<Q32Group> q32_host;          // fp32 path: [n_bd][kNLowRates]
  Q32Group* q32_dev = nullptr;

  // A bank whose chunk-local intermediates (y^s, rho^(d)) would force chunks shorter than kSplitChunk is cut at finalize into
  // PARTS: contiguous ranges of bins, each a bank of its own (plan, state, history) over the parent's uploaded arrays,
  // run one after the other on the caller's stream.  The parts share one set of chunk-local buffers (scratch[]), so each
  // can afford a chunk n_parts times longer.  A parent runs no kernels of its own.
  std::vector<lloid_bank*> parts;
  std::vector<int> part_of_bin;          // parent: part index of a bin
  lloid_bank* parent = nullptr;
  int bin_base = 0;                      // part: first bin of its range (added to the bin index of its triggers)
  double budget = 0.0;                   // part: bytes its chunk-local intermediates may take (the parent decides)
  struct Scratch { void* p = nullptr; size_t cap = 0; } scratch[3];   // parent: 0 y^s, 1 rho^(d) (fp16 plan), 2 partial peaks

  int slice_index(int bin, int det, int s) const { return bp_host[bin * cfg.n_detectors + det].first_slice + s; }
};

namespace {

int dev_alloc(lloid_bank* b, void** p, size_t n, bool zero)
{
  if (n == 0) n = 16;
  cudaError_t e = cudaMalloc(p, n);
  if (e != cudaSuccess) return fail(LLOID_ENOMEM, "cudaMalloc(%zu) failed: %s", n, cudaGetErrorString(e));
  if (zero) { e = cudaMemset(*p, 0, n); if (e != cudaSuccess) return fail(LLOID_ECUDA, "cudaMemset: %s", cudaGetErrorString(e)); }
  b->owned.push_back(*p);
  b->bytes += (int64_t)n;
  return LLOID_OK;
}

// Chunk-local buffers (kind: 0 y^s, 1 rho^(d), 2 partial peaks).  A whole bank allocates its own.  A part takes them from
// its parent's shared set: every part's buffer of a kind starts at the same address -- fp16 data over fp16 data, records
// over records, so whatever an earlier part left there is finite -- and the parts never run concurrently.
int scratch_alloc(lloid_bank* b, int kind, void** p, size_t n, bool zero)
{
  if (!b->parent) return dev_alloc(b, p, n, zero);
  lloid_bank::Scratch& S = b->parent->scratch[kind];
  if (n > S.cap) {
    const size_t want = n + n / 32;                  // the parts are finalized largest first; headroom for padding differences
    void* q = nullptr;
    int rc = dev_alloc(b->parent, &q, want, true);   // (an outgrown buffer stays with the parts that point into it)
    if (rc) return rc;
    S.p = q; S.cap = want;
  }
  *p = S.p;
  return LLOID_OK;
}

void* plan_scratch_alloc(void* ctx, size_t n)
{
  void* p = nullptr;
  return scratch_alloc((lloid_bank*)ctx, 1, &p, n, true) == LLOID_OK ? p : nullptr;
}

int upload_arrays(lloid_bank* b, int bin, int slice, const double* basis, const double* recon,
                  const float** U32, const float** R32, const __half** U16, const __half** U16b, const __half** R16)
{
  const BinHost& B = b->bins[bin];
  const SliceHost& S = B.slices[slice];
  const size_t nu = (size_t)S.L_pad * S.n_taps, nr = (size_t)B.rows_pad * S.L_pad;
  *U32 = nullptr; *R32 = nullptr; *U16 = nullptr; *U16b = nullptr; *R16 = nullptr;
  if (!b->f16) {
    std::vector<float> u(nu, 0.f), r(nr, 0.f);
    for (int l = 0; l < S.L; ++l)
      for (int t = 0; t < S.n_taps; ++t) u[(size_t)l * S.n_taps + t] = (float)basis[(size_t)l * S.n_taps + t];
    for (int i = 0; i < 2 * B.N; ++i)
      for (int l = 0; l < S.L; ++l) r[(size_t)i * S.L_pad + l] = (float)recon[(size_t)i * S.L + l];
    void *du, *dr;
    int rc = dev_alloc(b, &du, nu * 4, false); if (rc) return rc;
    rc = dev_alloc(b, &dr, nr * 4, false); if (rc) return rc;
    CU(cudaMemcpy(du, u.data(), nu * 4, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(dr, r.data(), nr * 4, cudaMemcpyHostToDevice));
    *U32 = (const float*)du; *R32 = (const float*)dr;
  } else {
    // fp16 path: U packed for the tcgen05 FIR kernel as [tap block of 64][tap group of 8][l < L_pad][8 taps]
    // (taps zero-padded to a multiple of 64); R packed as R16[i / 128][l / 8][r16_lane(i % 128)][l % 8]
    // (lloid_internal.h): a reconstruction CTA bulk-copies its 128-row block straight into MMA layout.
    // A folded slice (lloid_internal.h, kFoldMaxD) stores, per output phase phi, Uhat_phi[l, u] = sum_i w_phi[i] U[l, u - K_up + i]
    // with n_s + 2 K_up taps (w_phi[i] = d lp_{d,K_up}[d i + phi], i = -K_up .. K_up - 1), computed in double precision.
    const int Ku = b->cfg.k_up;
    const int n_eff = S.fold ? S.n_taps + 2 * Ku : S.n_taps;
    const int n_kb = (n_eff + 63) / 64;
    const size_t nup = (size_t)n_kb * 64 * S.L_pad;
    std::vector<__half> u(nup, __float2half(0.f)), ub;
    auto upos = [&](int l, int t) {            // column block of l, then [tap block][tap group][l in block][8 taps]
      int bi = 0;
      while (bi + 1 < S.n_ub && l >= S.ub_l0[bi + 1]) ++bi;
      return S.ub_off(bi, n_kb) + (((size_t)(t >> 6) * 8 + ((t >> 3) & 7)) * S.ub_w[bi] + (l - S.ub_l0[bi])) * 8 + (t & 7);
    };
    if (!S.fold) {
      for (int l = 0; l < S.L; ++l)
        for (int t = 0; t < S.n_taps; ++t)
          u[upos(l, t)] = __float2half_rn((float)basis[(size_t)l * S.n_taps + t]);
    } else {
      ub.assign(nup, __float2half(0.f));
      const std::vector<double> lp = lowpass(S.d, Ku);
      for (int phi = 0; phi < 2; ++phi) {
        std::vector<__half>& dst = phi ? ub : u;
        for (int l = 0; l < S.L; ++l)
          for (int uu = 0; uu < n_eff; ++uu) {
            double acc = 0.0;
            for (int i = -Ku; i < Ku; ++i) {
              const int t = uu - Ku + i;
              if (t < 0 || t >= S.n_taps) continue;
              acc += (double)S.d * lp[S.d * i + phi + Ku * S.d] * basis[(size_t)l * S.n_taps + t];
            }
            dst[upos(l, uu)] = __float2half_rn((float)acc);
          }
      }
    }
    std::vector<__half> r(nr, __float2half(0.f));
    const size_t lgs = (size_t)(S.L_pad >> 3);
    for (int i = 0; i < 2 * B.N; ++i)
      for (int l = 0; l < S.L; ++l)
        r[(((size_t)(i >> 7) * lgs + (l >> 3)) * 128 + r16_lane(i & 127)) * 8 + (l & 7)] =
            __float2half_rn((float)recon[(size_t)i * S.L + l]);
    void *du, *dr;
    int rc = dev_alloc(b, &du, nup * 2, false); if (rc) return rc;
    rc = dev_alloc(b, &dr, nr * 2, false); if (rc) return rc;
    CU(cudaMemcpy(du, u.data(), nup * 2, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(dr, r.data(), nr * 2, cudaMemcpyHostToDevice));
    *U16 = (const __half*)du; *R16 = (const __half*)dr;
    if (S.fold) {
      void* dub;
      rc = dev_alloc(b, &dub, nup * 2, false); if (rc) return rc;
      CU(cudaMemcpy(dub, ub.data(), nup * 2, cudaMemcpyHostToDevice));
      *U16b = (const __half*)dub;
    }
  }
  return LLOID_OK;
}

int check_ids(const lloid_bank* b, int bin, int det, int slice)
{
  if (!b) return fail(LLOID_EINVAL, "null bank");
  if (bin < 0 || bin >= b->cfg.n_bins) return fail(LLOID_EINVAL, "bin %d out of range", bin);
  if (det < 0 || det >= b->cfg.n_detectors) return fail(LLOID_EINVAL, "detector %d out of range", det);
  if (slice < 0 || slice >= b->bins[bin].S) return fail(LLOID_EINVAL, "slice %d out of range", slice);
  return LLOID_OK;
}

// profiling: the time between two consecutive events is charged to the stage tag of the later one
enum { kTagStart = -1, kTagResample = 0, kTagFir = 1, kTagRecon = 2, kTagMerge = 3, kTagLowRecon = 5 };
cudaEvent_t grab(lloid_bank* b, int tag)          // next event of the list, tagged; the caller records it
{
  if (!b->prof) return nullptr;
  if (b->events_used == b->events.size()) {
    cudaEvent_t e; cudaEventCreate(&e); b->events.push_back(e); b->event_tag.push_back(tag);
  }
  b->event_tag[b->events_used] = tag;
  return b->events[b->events_used++];
}
void mark(lloid_bank* b, cudaStream_t st, int tag)
{
  if (cudaEvent_t e = grab(b, tag)) cudaEventRecord(e, st);
}

// A1 for one super-chunk [k_s, k_s + n_s): xw = [history | strain], new history saved, every rate resampled once.
int stage_superchunk(lloid_bank* b, const float* strain, int64_t pitch, int n_s, cudaStream_t st)
{
  const int D = b->cfg.n_detectors;
  const size_t wp = (size_t)b->xw_pitch * 4;
  CU(cudaMemcpy2DAsync(b->xw, wp, b->hist, (size_t)b->H * 4, (size_t)b->H * 4, D, cudaMemcpyDeviceToDevice, st));
  CU(cudaMemcpy2DAsync(b->xw + b->H, wp, strain, (size_t)pitch * 4, (size_t)n_s * 4, D, cudaMemcpyDeviceToDevice, st));
  CU(cudaMemcpy2DAsync(b->hist, (size_t)b->H * 4, b->xw + n_s, wp, (size_t)b->H * 4, D, cudaMemcpyDeviceToDevice, st));
  mark(b, st, kTagStart);
  launch_resample(b->rates_dev, b->rates_host.data(), (int)b->rates_host.size(), b->xw, b->xw_pitch,
                  b->H + n_s, D, b->cfg.k_down, n_s, b->f16, st, &b->last_launches);
  mark(b, st, kTagResample);
  return LLOID_OK;
}

// LLOID_DEBUG_SYNC=1 in the environment: synchronise after every kernel of a chunk and name the one that faulted
// (debugging aid only; lloid_filter is then no longer asynchronous).
int debug_sync(const char* what, int64_t k_a, cudaStream_t st)
{
  static const bool on = getenv("LLOID_DEBUG_SYNC") != nullptr;
  if (!on) return LLOID_OK;
  const cudaError_t e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail(LLOID_ECUDA, "%s faulted in the chunk starting at sample %lld: %s", what, (long long)k_a, cudaGetErrorString(e));
  return LLOID_OK;
}

// A2..A6 for one chunk [k_a, k_a + c) that starts `o` samples into the current super-chunk
int process_chunk(lloid_bank* b, int o, int c, int64_t k_a, lloid_trigger_t* trig, int64_t capacity,
                  unsigned long long* count, cudaStream_t st)
{
  const int D = b->cfg.n_detectors;
  const int n_prob = (int)b->sp_host.size();
  if (!b->f16) {
    launch_fir_f32(b->sp_dev, b->sp_host.data(), n_prob, b->rates_dev, D, o, c, st, &b->last_launches);
    mark(b, st, kTagFir);
    if (b->q32_dev) {
      launch_lowrate_gemm_f32(b->sp_dev, b->q32_dev, b->q32_host.data(), (int)b->q32_host.size(), b->max_rows_pad, c, false, st,
                              &b->last_launches);
      mark(b, st, kTagLowRecon);
      launch_recon_f32_q(b->sp_dev, b->bp_dev, b->n_bd, b->max_rows_pad, b->upw_dev, b->q32_dev, b->partials, b->slots_cap,
                         b->max_templates, c, k_a, b->cap, false, st, &b->last_launches);
    } else {
      launch_recon_f32(b->sp_dev, b->bp_dev, b->bp_host.data(), b->n_bd, b->max_rows_pad, b->upw_dev,
                       b->partials, b->slots_cap, b->max_templates, c, k_a, b->cap, false, st, &b->last_launches);
    }
  } else {
    if (launch_fir_f16(b->plan16, b->fir_dev, b->fir_host.data(), (int)b->fir_host.size(), b->rates_dev, o, c, st, &b->last_launches))
      return fail(LLOID_ECUDA, "fp16 FIR launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    mark(b, st, kTagFir);
    if (int rc = debug_sync("fir_f16_kernel", k_a, st)) return rc;
    if (f16_plan_tensor_recon(b->plan16)) {
      if (launch_recon_f16(b->plan16, b->sp_dev, b->partials, b->slots_cap, b->max_templates, c, k_a, b->gt, b->cfg.snr_threshold, b->cap, st,
                           &b->last_launches, grab(b, kTagLowRecon)))
        return fail(LLOID_ECUDA, "fp16 reconstruction launch failed: %s", cudaGetErrorString(cudaGetLastError()));
      if (b->q32_dev) {                              // mixed bank: the bins outside the tensor kernels' limits
        launch_lowrate_gemm_f32(b->sp_dev, b->q32_dev, b->q32_host.data(), (int)b->q32_host.size(), b->max_rows_pad, c, true, st,
                                &b->last_launches);
        launch_recon_f32_q(b->sp_dev, b->bp_dev, b->n_bd, b->max_rows_pad, b->upw_dev, b->q32_dev, b->partials, b->slots_cap,
                           b->max_templates, c, k_a, b->cap, true, st, &b->last_launches);
      }
    } else if (b->q32_dev) {
      // geometry the tensor reconstruction cannot hold: FFMA kernels of the fp32 path reading the
      // packed fp16 y and R (3.6x faster than the single fused CUDA-core kernel on the config-4 geometry)
      launch_lowrate_gemm_f32(b->sp_dev, b->q32_dev, b->q32_host.data(), (int)b->q32_host.size(), b->max_rows_pad, c, true, st,
                              &b->last_launches);
      mark(b, st, kTagLowRecon);
      launch_recon_f32_q(b->sp_dev, b->bp_dev, b->n_bd, b->max_rows_pad, b->upw_dev, b->q32_dev, b->partials, b->slots_cap,
                         b->max_templates, c, k_a, b->cap, true, st, &b->last_launches);
    } else {
      launch_recon_f32(b->sp_dev, b->bp_dev, b->bp_host.data(), b->n_bd, b->max_rows_pad, b->upw_dev,
                       b->partials, b->slots_cap, b->max_templates, c, k_a, b->cap, true, st, &b->last_launches);
    }
  }
  mark(b, st, kTagRecon);
  if (int rc = debug_sync("reconstruction kernels", k_a, st)) return rc;
  const size_t nstate = (size_t)b->n_bd * b->max_templates;
  launch_merge_windows(b->bp_dev, b->n_bd, b->max_templates, b->partials, b->slots_cap, b->slot_tiles_dev, c, k_a, b->k_base_dev, k_a - b->call_start,
                       b->cfg.peak_window, b->cfg.snr_threshold, b->state + b->state_cur * nstate,
                       b->state + (b->state_cur ^ 1) * nstate, D, b->bin_base, trig, capacity, count, st, &b->last_launches);
  b->state_cur ^= 1;
  mark(b, st, kTagMerge);
  if (int rc = debug_sync("merge_windows_kernel", k_a, st)) return rc;
  CU(cudaGetLastError());
  return LLOID_OK;
}

}  // namespace

extern "C" {

const char* lloid_last_error(void) { return g_err.c_str(); }
const char* lloid_version(void) { return "lloid-b200 0.1 (sm_100a)"; }

int lloid_check_count(int64_t count, int64_t capacity)
{
  if (count > capacity) return fail(LLOID_EOVERFLOW, "trigger buffer overflow: %lld triggers, capacity %lld",
                                    (long long)count, (long long)capacity);
  return LLOID_OK;
}

int lloid_bank_create(lloid_bank_t** out, const lloid_bank_config_t* cfg, const lloid_bin_desc_t* bins,
                      const lloid_slice_desc_t* const* slices)
{
  if (!out || !cfg || !bins || !slices) return fail(LLOID_EINVAL, "null argument");
  *out = nullptr;
  if (cfg->n_bins < 1 || cfg->n_detectors < 1) return fail(LLOID_EINVAL, "n_bins and n_detectors must be >= 1");
  if (cfg->full_rate_hz < 1) return fail(LLOID_EINVAL, "full_rate_hz must be positive");
  if (cfg->peak_window < kTimeTile || cfg->peak_window % kTimeTile)
    return fail(LLOID_EINVAL, "peak_window must be a positive multiple of %d", kTimeTile);
  if (cfg->k_up != kKUp) return fail(LLOID_EINVAL, "k_up must be %d in this version", kKUp);
  if (cfg->k_down < 1 || cfg->k_down > 64) return fail(LLOID_EINVAL, "k_down out of range [1, 64]");
  if (cfg->precision != LLOID_F32 && cfg->precision != LLOID_F16)
    return fail(LLOID_EINVAL, "precision must be LLOID_F32 or LLOID_F16");
  if (cfg->max_chunk < 0 || cfg->max_chunk % kTimeTile) return fail(LLOID_EINVAL, "max_chunk must be a multiple of %d", kTimeTile);
  if (!(cfg->snr_threshold >= 0.f)) return fail(LLOID_EINVAL, "snr_threshold must be >= 0");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(LLOID_ECUDA, "no CUDA device: this library has no CPU fallback");
  if (cfg->device < 0 || cfg->device >= ndev) return fail(LLOID_ECUDA, "device %d not present", cfg->device);
  cudaDeviceProp prop;
  CU(cudaGetDeviceProperties(&prop, cfg->device));
  if (prop.major != 10) return fail(LLOID_ECUDA, "device %d is sm_%d%d; this build is sm_100a only", cfg->device, prop.major, prop.minor);
  CU(cudaSetDevice(cfg->device));

  lloid_bank* b = new (std::nothrow) lloid_bank();
  if (!b) return fail(LLOID_ENOMEM, "out of host memory");
  b->cfg = *cfg;
  b->f16 = cfg->precision == LLOID_F16;
  b->bins.resize(cfg->n_bins);
  int first = 0;
  for (int bi = 0; bi < cfg->n_bins; ++bi) {
    const lloid_bin_desc_t& bd = bins[bi];
    BinHost& B = b->bins[bi];
    if (bd.n_templates < 1 || bd.n_slices < 1 || bd.template_len < 1 || !slices[bi]) {
      delete b; return fail(LLOID_EINVAL, "bin %d: bad descriptor", bi);
    }
    B.N = bd.n_templates; B.S = bd.n_slices; B.M = bd.template_len;
    B.rows_pad = (int)round_up(2 * B.N, b->f16 ? kRowPad16 : kRowPad);
    int64_t expect_delay = 0;
    for (int s = 0; s < B.S; ++s) {
      const lloid_slice_desc_t& sd = slices[bi][s];
      SliceHost S;
      if (sd.rate_hz < 1 || cfg->full_rate_hz % sd.rate_hz) { delete b; return fail(LLOID_EINVAL, "bin %d slice %d: rate %d does not divide f0", bi, s, sd.rate_hz); }
      S.rate = sd.rate_hz; S.d = cfg->full_rate_hz / sd.rate_hz; S.log2d = ilog2(S.d);
      if ((1 << S.log2d) != S.d || S.d > 32) { delete b; return fail(LLOID_EINVAL, "bin %d slice %d: decimation %d is not a power of two <= 32", bi, s, S.d); }
      if (sd.n_taps < 1 || sd.n_basis < 1 || sd.n_basis > 512) { delete b; return fail(LLOID_EINVAL, "bin %d slice %d: n_taps/n_basis out of range", bi, s); }
      if (sd.end_delay % S.d) { delete b; return fail(LLOID_EINVAL, "bin %d slice %d: end_delay not a multiple of d", bi, s); }
      if (sd.end_delay != expect_delay) { delete b; return fail(LLOID_EINVAL, "bin %d slice %d: slices must tile the template back to front (end_delay %lld, expected %lld)", bi, s, (long long)sd.end_delay, (long long)expect_delay); }
      if (S.d > 1 && sd.end_delay < (int64_t)(cfg->k_down + cfg->k_up) * S.d) { delete b; return fail(LLOID_EINVAL, "bin %d slice %d: causality needs end_delay >= (k_down + k_up) * d", bi, s); }
      S.n_taps = sd.n_taps; S.L = sd.n_basis; S.L_pad = (int)round_up(S.L, kLPad); S.end_delay = sd.end_delay;
      S.fold = b->f16 && S.d > 1 && S.d <= kFoldMaxD && !getenv("LLOID_NO_FOLD");
      S.set_blocks(b->f16);
      expect_delay += (int64_t)S.d * S.n_taps;
      B.slices.push_back(S);
      b->d_max = std::max(b->d_max, S.d);
    }
    if (expect_delay != B.M) { delete b; return fail(LLOID_EINVAL, "bin %d: slices cover %lld samples, template_len is %lld", bi, (long long)expect_delay, (long long)B.M); }
    {
      // folded slices are reconstructed at f0 next to the d = 1 slices: their summed L_pad must fit the f0 kernel's
      // stationary operand (512 basis filters); otherwise the bin keeps its low-rate slices on the low-rate path
      int l_f0 = 0, n_f0 = 0;
      for (const SliceHost& S : B.slices) if (S.d == 1 || S.fold) { l_f0 += S.L_pad; ++n_f0; }
      if (l_f0 > 512 || n_f0 > kMaxF0Slices) for (SliceHost& S : B.slices) S.fold = false;
    }
    b->max_templates = std::max(b->max_templates, B.N);
    b->max_rows_pad = std::max(b->max_rows_pad, B.rows_pad);
    for (int det = 0; det < cfg->n_detectors; ++det) {
      BinParams bp; bp.n_templates = B.N; bp.n_slices = B.S; bp.first_slice = first; bp.rows_pad = B.rows_pad;
      b->bp_host.push_back(bp);
      for (int s = 0; s < B.S; ++s) {
        SliceParams P; memset(&P, 0, sizeof P);
        const SliceHost& S = B.slices[s];
        P.d = S.fold ? 1 : S.d; P.log2d = S.fold ? 0 : S.log2d; P.n_taps = S.n_taps; P.L = S.L; P.L_pad = S.L_pad;   // reconstruction view
        P.rows = 2 * B.N; P.rows_pad = B.rows_pad; P.bin = bi; P.det = det; P.slice = s;
        b->sp_host.push_back(P);
      }
      first += B.S;
    }
  }
  b->n_bd = cfg->n_bins * cfg->n_detectors;
  b->uploaded.assign(b->sp_host.size(), 0);
  *out = b;
  return LLOID_OK;
}

int lloid_bank_upload_slice(lloid_bank_t* b, int32_t bin, int32_t det, int32_t slice, const double* basis,
                            const double* recon)
{
  int rc = check_ids(b, bin, det, slice); if (rc) return rc;
  if (!basis || !recon) return fail(LLOID_EINVAL, "null array");
  if (b->finalized) return fail(LLOID_ESTATE, "upload after finalize");
  CU(cudaSetDevice(b->cfg.device));
  SliceParams& P = b->sp_host[b->slice_index(bin, det, slice)];
  rc = upload_arrays(b, bin, slice, basis, recon, &P.U32, &P.R32, &P.U16, &P.U16b, &P.R16); if (rc) return rc;
  b->uploaded[b->slice_index(bin, det, slice)] = 1;
  return LLOID_OK;
}

int lloid_bank_upload_slice_shared(lloid_bank_t* b, int32_t bin, int32_t slice, const double* basis,
                                   const double* recon)
{
  int rc = check_ids(b, bin, 0, slice); if (rc) return rc;
  if (!basis || !recon) return fail(LLOID_EINVAL, "null array");
  if (b->finalized) return fail(LLOID_ESTATE, "upload after finalize");
  CU(cudaSetDevice(b->cfg.device));
  SliceParams& P0 = b->sp_host[b->slice_index(bin, 0, slice)];
  rc = upload_arrays(b, bin, slice, basis, recon, &P0.U32, &P0.R32, &P0.U16, &P0.U16b, &P0.R16); if (rc) return rc;
  for (int det = 0; det < b->cfg.n_detectors; ++det) {
    SliceParams& P = b->sp_host[b->slice_index(bin, det, slice)];
    P.U32 = P0.U32; P.R32 = P0.R32; P.U16 = P0.U16; P.U16b = P0.U16b; P.R16 = P0.R16;
    b->uploaded[b->slice_index(bin, det, slice)] = 1;
  }
  return LLOID_OK;
}

int lloid_bank_alias_bin(lloid_bank_t* b, int32_t dst, int32_t src)
{
  int rc = check_ids(b, dst, 0, 0); if (rc) return rc;
  rc = check_ids(b, src, 0, 0); if (rc) return rc;
  if (b->finalized) return fail(LLOID_ESTATE, "alias after finalize");
  const BinHost &A = b->bins[dst], &Bs = b->bins[src];
  if (A.N != Bs.N || A.S != Bs.S || A.M != Bs.M) return fail(LLOID_EINVAL, "alias_bin: geometry differs");
  for (int s = 0; s < A.S; ++s) {
    const SliceHost &x = A.slices[s], &y = Bs.slices[s];
    if (x.d != y.d || x.n_taps != y.n_taps || x.L != y.L || x.end_delay != y.end_delay)
      return fail(LLOID_EINVAL, "alias_bin: slice %d geometry differs", s);
    for (int det = 0; det < b->cfg.n_detectors; ++det) {
      const int is = b->slice_index(src, det, s), id = b->slice_index(dst, det, s);
      if (!b->uploaded[is]) return fail(LLOID_ESTATE, "alias_bin: source bin %d not uploaded", src);
      SliceParams& P = b->sp_host[id]; const SliceParams& Q = b->sp_host[is];
      P.U32 = Q.U32; P.R32 = Q.R32; P.U16 = Q.U16; P.U16b = Q.U16b; P.R16 = Q.R16;
      b->uploaded[id] = 1;
    }
  }
  return LLOID_OK;
}

}  // extern "C"

namespace {

constexpr int64_t kSplitChunk = 32768;   // a bank whose automatic chunk would be shorter than this is cut into parts

// bytes of chunk-local intermediates per f0 sample of bins [lo, hi): y^s of every slice, rho^(d) of the low-rate ones
double intermediates_per_sample(const lloid_bank* b, int lo, int hi)
{
  const int D = b->cfg.n_detectors;
  const size_t esize = b->f16 ? 2 : 4;
  double v = 0.0;
  for (int bi = lo; bi < hi; ++bi) {
    const BinHost& B = b->bins[bi];
    for (const SliceHost& S : B.slices) {
      v += (double)D * S.L_pad * esize / (S.fold ? 1 : S.d);
      if (S.d > 1 && !S.fold) v += (double)D * B.rows_pad * esize / S.d;
    }
  }
  return v;
}

int finalize_impl(lloid_bank* b);
int filter_one(lloid_bank* b, const float* strain_dev, int64_t n, lloid_trigger_t* trig, int64_t capacity, int64_t* count_dev, cudaStream_t st);

// a part: bins [lo, hi) of the parent as a bank of its own over the parent's device arrays
lloid_bank* make_part(lloid_bank* parent, int lo, int hi, double budget)
{
  lloid_bank* c = new (std::nothrow) lloid_bank();
  if (!c) return nullptr;
  c->cfg = parent->cfg; c->cfg.n_bins = hi - lo;
  c->f16 = parent->f16; c->parent = parent; c->bin_base = lo; c->budget = budget;
  c->bins.assign(parent->bins.begin() + lo, parent->bins.begin() + hi);
  const int D = parent->cfg.n_detectors;
  int first = 0;
  for (int bi = lo; bi < hi; ++bi) {
    const BinHost& B = parent->bins[bi];
    c->max_templates = std::max(c->max_templates, B.N);
    c->max_rows_pad = std::max(c->max_rows_pad, B.rows_pad);
    for (const SliceHost& S : B.slices) c->d_max = std::max(c->d_max, S.d);
    for (int det = 0; det < D; ++det) {
      BinParams bp = parent->bp_host[(size_t)bi * D + det];
      const int src = bp.first_slice;
      bp.first_slice = first;
      c->bp_host.push_back(bp);
      for (int s = 0; s < B.S; ++s) {
        SliceParams P = parent->sp_host[src + s];
        P.bin = bi - lo;
        c->sp_host.push_back(P);
      }
      first += B.S;
    }
  }
  c->n_bd = (hi - lo) * D;
  c->uploaded.assign(c->sp_host.size(), 1);
  return c;
}

}  // namespace

extern "C" {

int lloid_bank_finalize(lloid_bank_t* b)
{
  if (!b) return fail(LLOID_EINVAL, "null bank");
  if (b->finalized) return fail(LLOID_ESTATE, "already finalized");
  for (size_t i = 0; i < b->uploaded.size(); ++i)
    if (!b->uploaded[i]) return fail(LLOID_ESTATE, "bin %d detector %d slice %d was never uploaded",
                                     b->sp_host[i].bin, b->sp_host[i].det, b->sp_host[i].slice);
  CU(cudaSetDevice(b->cfg.device));
  // Split?  fp16 path with automatic chunking only, when memory (not the 2^17 cap) would bound the chunk below kSplitChunk.
  const int n_bins = b->cfg.n_bins;
  if (b->f16 && b->cfg.max_chunk == 0 && n_bins >= 2 && !getenv("LLOID_NO_SPLIT")) {
    size_t mem_free = 0, mem_total = 0;
    CU(cudaMemGetInfo(&mem_free, &mem_total));
    double budget = 0.5 * (double)mem_free;
    budget = std::min(std::max(budget, 4.0 * 1024 * 1024 * 1024), 96.0 * 1024 * 1024 * 1024);
    const double per_sample = intermediates_per_sample(b, 0, n_bins);
    int n_parts = 1;
    if (getenv("LLOID_PARTS")) n_parts = atoi(getenv("LLOID_PARTS"));                    // tests and A/B measurements
    else if (budget / per_sample < (double)kSplitChunk) n_parts = (int)std::ceil(per_sample * (double)kSplitChunk / budget);
    n_parts = std::max(1, std::min(n_parts, n_bins));
    if (n_parts > 1) {
      // contiguous ranges of bins with (nearly) equal shares of the intermediates, at least one bin each
      std::vector<double> cum(n_bins + 1, 0.0);
      for (int bi = 0; bi < n_bins; ++bi) cum[bi + 1] = cum[bi] + intermediates_per_sample(b, bi, bi + 1);
      int lo = 0;
      for (int part = 0; part < n_parts; ++part) {
        int hi = lo + 1;
        const int hi_max = n_bins - (n_parts - 1 - part);            // leave one bin for every part still to come
        while (hi < hi_max && cum[hi + 1] <= cum[n_bins] * (part + 1) / n_parts * (1.0 + 1e-9)) ++hi;
        if (part == n_parts - 1) hi = n_bins;
        lloid_bank* c = make_part(b, lo, hi, budget);
        if (!c) return fail(LLOID_ENOMEM, "out of host memory");
        b->parts.push_back(c);
        for (int bi = lo; bi < hi; ++bi) b->part_of_bin.push_back(part);
        lo = hi;
      }
      // largest first: the shared chunk-local buffers are sized by the first part that asks
      std::vector<int> order(n_parts);
      for (int i = 0; i < n_parts; ++i) order[i] = i;
      std::sort(order.begin(), order.end(), [&](int x, int y) {
        const lloid_bank *X = b->parts[x], *Y = b->parts[y];
        return cum[X->bin_base + X->cfg.n_bins] - cum[X->bin_base] > cum[Y->bin_base + Y->cfg.n_bins] - cum[Y->bin_base];
      });
      for (int i : order) {
        const int rc = finalize_impl(b->parts[i]);
        if (rc) return rc;
      }
      b->C = b->parts[0]->C; b->H = b->parts[0]->H; b->S = b->parts[0]->S;
      for (const lloid_bank* c : b->parts) { b->C = std::min(b->C, c->C); b->H = std::max(b->H, c->H); }
      int rc = dev_alloc(b, (void**)&b->stage_count, 8, true); if (rc) return rc;
      b->finalized = true;
      return LLOID_OK;
    }
  }
  return finalize_impl(b);
}

}  // extern "C"

namespace {

int finalize_impl(lloid_bank* b)
{
  CU(cudaSetDevice(b->cfg.device));
  const int D = b->cfg.n_detectors, Kd = b->cfg.k_down, Ku = b->cfg.k_up;
  const size_t esize = b->f16 ? 2 : 4;

  // history length H: enough strain before the chunk for every slice's earliest tap
  int64_t H = 0;
  double ybytes_per_sample = 0.0;
  for (const BinHost& B : b->bins)
    for (const SliceHost& S : B.slices) {
      const int64_t need = (S.d == 1) ? S.end_delay + S.n_taps : S.end_delay + (int64_t)S.d * (S.n_taps + Ku + Kd);
      H = std::max(H, need);
      ybytes_per_sample += (double)D * S.L_pad * esize / (S.fold ? 1 : S.d);
      if (S.d > 1 && !S.fold) ybytes_per_sample += (double)D * B.rows_pad * esize / S.d;   // rho^(d) staging (upper bound)
    }
  H = round_up(H, 256);
  if (H > (1ll << 28)) return fail(LLOID_EINVAL, "history too long");
  int64_t C = b->cfg.max_chunk;
  size_t mem_free = 0, mem_total = 0;
  CU(cudaMemGetInfo(&mem_free, &mem_total));
  if (C == 0) {
    // Every chunk costs four kernel boundaries (launch gap, prologue with TMEM allocation and the stationary
    // operands, pipeline fill and drain), and every low-rate slice computes 2 K_up halo rows and rounds its rows up to
    // 128-row MMA tiles per chunk, so chunks are made LONG: up to 2^17 samples, bounded by the chunk-local
    // intermediates (y^s and the low-rate rho^(d)), which may take half of the free device memory (4 ... 96 GiB).
    // BASELINE config 2 (2 (bin, detector) pairs): 131072 samples = 1.2 GB; config 4 (3000 pairs): 7680 samples = 60 GB.
    double budget = 0.5 * (double)mem_free;
    budget = std::min(std::max(budget, 4.0 * 1024 * 1024 * 1024), 96.0 * 1024 * 1024 * 1024);
    if (b->parent) budget = b->budget;                    // a part: the parent's figure (the parts share the buffers)
    C = (int64_t)(budget / ybytes_per_sample) / 2048 * 2048;
    C = std::min<int64_t>(std::max<int64_t>(C, 2048), 131072);
    if (b->f16 && C < 32768) {
      // A memory-bound chunk is short, and then the 128-row MMA tiles of the low rates matter: a slice at f0 / d computes
      // ceil((C / d + 2 K_up) / 128) tiles per chunk (C = 6144, d = 32: 208 rows in 2 tiles, 19 % padding; C = 7680: 256
      // rows, none).  Take the multiple of 128 in (C_max / 2, C_max] with the least padded tensor work per sample.
      const int64_t c_max = std::min<int64_t>((int64_t)(budget / ybytes_per_sample) / 128 * 128, 131072);
      double best = 1e300;
      for (int64_t c = std::max<int64_t>(2048, c_max / 2 / 128 * 128); c <= c_max; c += 128) {
        double cost = 0.0;
        for (const BinHost& B : b->bins)
          for (const SliceHost& S : B.slices) {
            const double w = (double)S.L_pad * (S.n_taps + B.rows_pad) / S.d;          // MACs per f0 sample
            const double rows = (S.d == 1 || S.fold) ? (double)c : std::ceil(((double)c / S.d + 2 * Ku) / 128.0) * 128.0 * S.d;
            cost += w * rows;
          }
        cost /= (double)c;
        if (cost <= best * (1.0 + 1e-9)) { best = cost; C = c; }                       // ties: the longer chunk
      }
    }
  }
  {
    // the allocations below, estimated up front so that a bank that cannot fit fails with a message instead of a
    // cudaMalloc error half-way through (intermediates dominate; 128-row paddings and the halo included)
    double need = 0.0;
    for (const BinHost& B : b->bins)
      for (const SliceHost& S : B.slices) {
        const double rows = (S.d == 1 || S.fold) ? (double)C : (double)C / S.d + 2 * Ku;
        need += (double)D * (std::ceil(rows / 128.0) * 128.0) * S.L_pad * esize;
      }
    if (b->f16)
      for (const BinHost& B : b->bins) {
        bool seen[kMaxRates] = {false, false, false, false, false, false};
        for (const SliceHost& S : B.slices) {
          if (S.d == 1 || S.fold || seen[S.log2d]) continue;
          seen[S.log2d] = true;
          need += (double)D * ((std::ceil(((double)C / S.d + 2 * Ku) / 128.0) * 16 + 16) * 8) * B.rows_pad * 2.0;
        }
      }
    if (need > 0.95 * (double)mem_free + (b->parent ? (double)(b->parent->scratch[0].cap + b->parent->scratch[1].cap) : 0.0))
      return fail(LLOID_ENOMEM, "bank does not fit: chunk-local intermediates need %.1f GB at a chunk of %lld samples, %.1f GB of device memory are free "
                                "(reduce max_chunk, the number of bins per bank, or shard the bins over more GPUs)", need * 1e-9, (long long)C, (double)mem_free * 1e-9);
  }
  b->H = (int)H; b->C = (int)C;
  // A1 runs once per super-chunk of S samples (not per chunk): the strain is tiny (8 KB/s per detector), so a
  // long stretch of every rate stays resident and one launch streams it at HBM speed
  int64_t S = std::max<int64_t>(C, (int64_t)1 << 20);
  S = S / C * C;
  b->S = (int)S;
  b->xw_pitch = (int)round_up(H + S + 256, 64);
  b->tiles_cap = (int)(C / kTimeTile) + 1;

  int rc;
  rc = dev_alloc(b, (void**)&b->xw, (size_t)D * b->xw_pitch * 4, true); if (rc) return rc;
  rc = dev_alloc(b, (void**)&b->hist, (size_t)D * H * 4, true); if (rc) return rc;

  // rates
  std::vector<int> ds;
  for (const BinHost& B : b->bins) for (const SliceHost& S : B.slices) if (std::find(ds.begin(), ds.end(), S.d) == ds.end()) ds.push_back(S.d);
  std::sort(ds.begin(), ds.end());
  b->rates_host.resize(ds.size());
  for (size_t r = 0; r < ds.size(); ++r) {
    RateParams& R = b->rates_host[r]; memset(&R, 0, sizeof R);
    R.d = ds[r];
    R.jj_lo_fixed = INT32_MAX; R.jj_hi_off = INT32_MIN;
    if (R.d == 1) {
      R.xs32 = b->xw; R.xs_len = b->xw_pitch;
    } else {
      R.xs_len = (int)round_up((H + S) / R.d + 256, 64);
      rc = dev_alloc(b, (void**)&R.xs32, (size_t)D * R.xs_len * 4, true); if (rc) return rc;
      std::vector<double> lp = lowpass(R.d, Kd);
      std::vector<float> taps(lp.size());
      const double g = std::sqrt((double)R.d);
      for (size_t u = 0; u < lp.size(); ++u) taps[u] = (float)(g * lp[lp.size() - 1 - u]);
      float* td; rc = dev_alloc(b, (void**)&td, taps.size() * 4, false); if (rc) return rc;
      CU(cudaMemcpy(td, taps.data(), taps.size() * 4, cudaMemcpyHostToDevice));
      R.taps = td;
    }
    if (b->f16) { rc = dev_alloc(b, (void**)&R.xs16, (size_t)D * R.xs_len * 2, true); if (rc) return rc; }
  }

  // per-slice tables: Y buffers, origins, needed resample ranges
  size_t ybytes = 0;
  for (SliceParams& P : b->sp_host) {
    const SliceHost& S = b->bins[P.bin].slices[P.slice];
    P.rate_idx = (int)(std::find(ds.begin(), ds.end(), S.d) - ds.begin());      // the stream the FIR reads
    const int64_t rows = (S.d == 1 || S.fold) ? C : C / S.d + 2 * Ku;
    P.y_rows_cap = (int)round_up(rows, 128);
    // FIR window origin of Y row 0 (of FIR row 0 for a folded slice), in samples of the slice's rate stream
    P.jjY0 = (S.d == 1) ? (int)(H - S.end_delay) : (int)((H - S.end_delay) / S.d - Ku);
    P.fir_halo = (S.d == 1 || S.fold) ? 0 : 2 * Ku; P.out_mul = 1; P.out_add = 0;
    RateParams& R = b->rates_host[P.rate_idx];
    R.jj_lo_fixed = std::min(R.jj_lo_fixed, P.jjY0 - S.n_taps);
    R.jj_hi_off = std::max(R.jj_hi_off, (S.d == 1) ? P.jjY0 : P.jjY0 + 2 * Ku - 1);
    ybytes += round_up((size_t)P.y_rows_cap * S.L_pad * esize, 256);
  }
  char* ybase; rc = scratch_alloc(b, 0, (void**)&ybase, ybytes, true); if (rc) return rc;
  size_t yoff = 0;
  if (!b->f16) {
    for (SliceParams& P : b->sp_host) {
      P.Y = ybase + yoff; P.y_step64 = 0;
      yoff += round_up((size_t)P.y_rows_cap * P.L_pad * esize, 256);
    }
  } else {
    // Y16 is stored per RATE GROUP -- the slices of a (bin, detector) that are reconstructed at the same rate (a folded
    // slice counts as d = 1), in slice order: [64-row tile][slice][l / 8][64][8].  One 64-row tile of the whole group is one
    // contiguous record, so the reconstruction kernels stream a tile's K = sum L_pad operand with consecutive bulk copies.
    for (size_t i = 0; i < b->sp_host.size(); ++i) {
      SliceParams& P = b->sp_host[i];
      if (P.Y) continue;                                   // already placed with its group
      int rec = 0, rows_cap = 0;
      for (size_t j = i; j < b->sp_host.size() && b->sp_host[j].bin == P.bin && b->sp_host[j].det == P.det; ++j)
        if (b->sp_host[j].d == P.d) { rec += b->sp_host[j].L_pad * 128; rows_cap = std::max(rows_cap, b->sp_host[j].y_rows_cap); }
      int off = 0;
      for (size_t j = i; j < b->sp_host.size() && b->sp_host[j].bin == P.bin && b->sp_host[j].det == P.det; ++j) {
        SliceParams& Q = b->sp_host[j];
        if (Q.d != P.d) continue;
        Q.Y = ybase + yoff + off; Q.y_step64 = rec; Q.y_rows_cap = rows_cap;
        off += Q.L_pad * 128;
      }
      yoff += round_up((size_t)(rows_cap / 64) * rec, 256);
    }
    if (yoff > ybytes) return fail(LLOID_EINVAL, "internal: Y16 group layout exceeds its allocation");
  }
  for (const RateParams& R : b->rates_host)
    if (R.jj_lo_fixed < (R.d == 1 ? 0 : Kd)) return fail(LLOID_EINVAL, "internal: history too short for rate d=%d", R.d);
  if (b->f16) {
    // FIR problem table.  A folded slice (lloid_internal.h) contributes one problem per output phase: n_s + 2 K_up taps of
    // the composite filters, c / d rows, FIR row m -> Y row d m + phi; its window origin moves by the 2 K_up extra taps.
    for (const SliceParams& P : b->sp_host) {
      const SliceHost& S = b->bins[P.bin].slices[P.slice];
      const int n_phase = S.fold ? S.d : 1;
      const int n_kb = ((S.fold ? S.n_taps + 2 * Ku : S.n_taps) + 63) / 64;
      for (int phi = 0; phi < n_phase; ++phi) {
        SliceParams F = P;
        if (S.fold) {
          F.d = S.d; F.log2d = S.log2d; F.n_taps = S.n_taps + 2 * Ku; F.jjY0 = P.jjY0 + 2 * Ku;
          F.U16 = phi ? P.U16b : P.U16; F.fir_halo = 0; F.out_mul = S.d; F.out_add = phi;
        }
        for (int ub = 0; ub < S.n_ub; ++ub) {           // one problem per column block of the basis (SliceHost::set_blocks)
          SliceParams G = F;
          G.U16 = F.U16 + S.ub_off(ub, n_kb);
          G.L_pad = S.ub_w[ub]; G.L = std::max(0, std::min(S.L - S.ub_l0[ub], S.ub_w[ub]));
          G.Y = (char*)P.Y + (size_t)(S.ub_l0[ub] / 8) * 64 * 16;       // Y16 record: [slice][l / 8][64 rows][8]
          b->fir_host.push_back(G);
        }
      }
    }
    rc = dev_alloc(b, (void**)&b->fir_dev, b->fir_host.size() * sizeof(SliceParams), false); if (rc) return rc;
    CU(cudaMemcpy(b->fir_dev, b->fir_host.data(), b->fir_host.size() * sizeof(SliceParams), cudaMemcpyHostToDevice));
  }

  // interpolation weights  w[(i + K_up) * d + phi] = d * lp_{d,K_up}[d i + phi],  i = -K_up .. K_up - 1
  std::vector<const float*> upw(kMaxRates, nullptr);
  std::vector<std::vector<double>> upw64(kMaxRates);
  for (int d : ds) {
    if (d == 1) continue;
    std::vector<double> lp = lowpass(d, Ku);
    std::vector<float> w((size_t)2 * Ku * d);
    std::vector<double>& w64 = upw64[ilog2(d)];
    w64.resize(w.size());
    for (int i = -Ku; i < Ku; ++i)
      for (int phi = 0; phi < d; ++phi) {
        w64[(size_t)(i + Ku) * d + phi] = d * lp[d * i + phi + Ku * d];
        w[(size_t)(i + Ku) * d + phi] = (float)w64[(size_t)(i + Ku) * d + phi];
      }
    float* wd; rc = dev_alloc(b, (void**)&wd, w.size() * 4, false); if (rc) return rc;
    CU(cudaMemcpy(wd, w.data(), w.size() * 4, cudaMemcpyHostToDevice));
    upw[ilog2(d)] = wd;
  }
  rc = dev_alloc(b, (void**)&b->upw_dev, kMaxRates * sizeof(float*), false); if (rc) return rc;
  CU(cudaMemcpy((void*)b->upw_dev, upw.data(), kMaxRates * sizeof(float*), cudaMemcpyHostToDevice));

  rc = dev_alloc(b, (void**)&b->sp_dev, b->sp_host.size() * sizeof(SliceParams), false); if (rc) return rc;
  CU(cudaMemcpy(b->sp_dev, b->sp_host.data(), b->sp_host.size() * sizeof(SliceParams), cudaMemcpyHostToDevice));
  rc = dev_alloc(b, (void**)&b->bp_dev, b->bp_host.size() * sizeof(BinParams), false); if (rc) return rc;
  CU(cudaMemcpy(b->bp_dev, b->bp_host.data(), b->bp_host.size() * sizeof(BinParams), cudaMemcpyHostToDevice));
  rc = dev_alloc(b, (void**)&b->rates_dev, b->rates_host.size() * sizeof(RateParams), false); if (rc) return rc;
  CU(cudaMemcpy(b->rates_dev, b->rates_host.data(), b->rates_host.size() * sizeof(RateParams), cudaMemcpyHostToDevice));

  const size_t nstate = (size_t)b->n_bd * b->max_templates;
  rc = dev_alloc(b, (void**)&b->state, 2 * nstate * sizeof(PeakState), false); if (rc) return rc;
  rc = dev_alloc(b, (void**)&b->stage_count, 8, true); if (rc) return rc;
  rc = dev_alloc(b, (void**)&b->k_base_dev, 8, true); if (rc) return rc;
  launch_reset_state(b->state, 2 * (int64_t)nstate, 0);
  CU(cudaDeviceSynchronize());

  if (configure_common_kernels() || configure_f32_kernels()) return fail(LLOID_ECUDA, "cudaFuncSetAttribute failed: %s", cudaGetErrorString(cudaGetLastError()));
  if (b->f16) {
    char err[256] = {0};
    const double* up_w[kMaxRates];
    for (int l2 = 0; l2 < kMaxRates; ++l2) up_w[l2] = upw64[l2].empty() ? nullptr : upw64[l2].data();
    b->plan16 = f16_plan_create(b->sp_host.data(), (int)b->sp_host.size(), b->fir_host.data(), (int)b->fir_host.size(),
                                b->bp_host.data(), b->n_bd, D, b->C, up_w, b->parent ? plan_scratch_alloc : nullptr, b, &b->bytes, err, sizeof err);
    if (!b->plan16) return fail(LLOID_ECUDA, "fp16 plan: %s", err);
  }
  const uint8_t* excl = b->f16 ? f16_plan_excluded(b->plan16) : nullptr;   // mixed bank: only these bins use the FFMA kernels
  if (!b->f16 || !f16_plan_tensor_recon(b->plan16) || excl) {
    // fp32 path (and the fp16 path's CUDA-core fallback): one fp32 rho^(d) buffer per (bin, detector, low rate), filled
    // by lowrate_gemm_f32_kernel every chunk
    b->q32_host.assign((size_t)b->n_bd * kNLowRates, Q32Group());
    bool any = false, fits = true;
    for (int bd = 0; bd < b->n_bd; ++bd) {
      const BinParams& BP = b->bp_host[bd];
      for (int l2 = 1; l2 < kMaxRates; ++l2) {
        Q32Group& G = b->q32_host[(size_t)bd * kNLowRates + (l2 - 1)];
        memset(&G, 0, sizeof G);
        G.log2d = l2; G.rows_pad = BP.rows_pad; G.q_cols = (int)round_up((C >> l2) + 2 * Ku, 128);
        if (excl && !excl[bd]) { G.rows_pad = 0; continue; }     // reconstructed by the tensor kernels: both FFMA kernels skip it
        for (int s = 0; s < BP.n_slices; ++s)
          if (b->sp_host[BP.first_slice + s].log2d == l2) {
            if (G.n_slices == kMaxGroupSlices) { fits = false; break; }
            G.slice[G.n_slices++] = BP.first_slice + s;
          }
        if (G.n_slices) any = true;
      }
    }
    if ((any || excl) && fits) {
      for (Q32Group& G : b->q32_host)
        if (G.n_slices) { rc = dev_alloc(b, (void**)&G.Q, (size_t)G.rows_pad * G.q_cols * 4, true); if (rc) return rc; }
      rc = dev_alloc(b, (void**)&b->q32_dev, b->q32_host.size() * sizeof(Q32Group), false); if (rc) return rc;
      CU(cudaMemcpy(b->q32_dev, b->q32_host.data(), b->q32_host.size() * sizeof(Q32Group), cudaMemcpyHostToDevice));
    } else if (excl) {
      f16_plan_disable_tensor_recon(b->plan16);      // > 8 same-rate slices in an excluded bin: single fused CUDA-core kernel for the bank
    }
  }
  // partial peaks: the tensor kernels write one record per (template, granule of gt tiles), the CUDA-core kernels one
  // per tile; a mixed bank keeps per-tile slots for everyone and tells the merge kernel which rule a (bin, detector) uses
  {
    const bool tensor = b->f16 && f16_plan_tensor_recon(b->plan16);
    b->gt = tensor ? f16_granule_tiles(b->cfg.peak_window) : 1;
    const bool per_tile = !tensor || excl != nullptr;
    const int tensor_slots = 2 * ((int)(C / kTimeTile) / b->gt + 2);     // two records per granule (the f0 epilogue's two warp groups)
    b->slots_cap = !tensor ? b->tiles_cap : (per_tile ? std::max(b->tiles_cap, tensor_slots) : tensor_slots);
    rc = scratch_alloc(b, 2, (void**)&b->partials, nstate * b->slots_cap * sizeof(Peak), true); if (rc) return rc;
    if (tensor) {
      std::vector<int32_t> stl(b->n_bd, b->gt | (1 << 16));              // tiles per granule | two records per granule
      if (excl) for (int bd = 0; bd < b->n_bd; ++bd) if (excl[bd]) stl[bd] = 1;
      rc = dev_alloc(b, (void**)&b->slot_tiles_dev, stl.size() * sizeof(int32_t), false); if (rc) return rc;
      CU(cudaMemcpy(b->slot_tiles_dev, stl.data(), stl.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    }
  }
  b->finalized = true;
  return LLOID_OK;
}

}  // namespace

extern "C" {

int lloid_filter(lloid_bank_t* b, const float* strain_dev, int64_t n, lloid_trigger_t* trig, int64_t capacity,
                 int64_t* count_dev, void* stream)
{
  if (!b) return fail(LLOID_EINVAL, "null bank");
  if (!b->finalized) return fail(LLOID_ESTATE, "filter before finalize");
  if (!strain_dev || !count_dev || (capacity > 0 && !trig)) return fail(LLOID_EINVAL, "null buffer");
  if (n <= 0 || n % b->d_max) return fail(LLOID_EINVAL, "n_samples must be a positive multiple of %d", b->d_max);
  if (capacity < 0) return fail(LLOID_EINVAL, "negative capacity");
  cudaStream_t st = (cudaStream_t)stream;
  CU(cudaSetDevice(b->cfg.device));
  CU(cudaMemsetAsync(count_dev, 0, 8, st));
  if (!b->parts.empty()) {
    // split bank: the parts filter the same buffer one after the other and append to the same trigger list
    b->last_launches = 0;
    for (lloid_bank* c : b->parts) {
      const int rc = filter_one(c, strain_dev, n, trig, capacity, count_dev, st);
      if (rc) return rc;
      b->last_launches += c->last_launches;
    }
    b->consumed = b->parts[0]->consumed;
    return LLOID_OK;
  }
  return filter_one(b, strain_dev, n, trig, capacity, count_dev, st);
}

}  // extern "C"

namespace {

// one bank (or one part of a split bank): the caller has validated the arguments and cleared the count
int filter_one(lloid_bank* b, const float* strain_dev, int64_t n, lloid_trigger_t* trig, int64_t capacity, int64_t* count_dev, cudaStream_t st)
{
  b->last_launches = 0;
  b->events_used = 0;
  int64_t k = b->consumed, off = 0, rem = n;
  b->call_start = k;
  while (rem > 0) {
    const int n_s = (int)std::min<int64_t>(rem, b->S);
    int rc = stage_superchunk(b, strain_dev + off, n, n_s, st);
    if (rc) return rc;
    int o = 0;
    while (o < n_s) {
      int64_t c = std::min<int64_t>(n_s - o, b->C);
      const int64_t mis = (k + o) % kTimeTile;
      if (mis) c = std::min<int64_t>(c, kTimeTile - mis);   // re-align chunk starts to the tile grid
      rc = process_chunk(b, o, (int)c, k + o, trig, capacity, (unsigned long long*)count_dev, st);
      if (rc) return rc;
      o += (int)c;
    }
    k += n_s; off += n_s; rem -= n_s;
  }
  launch_advance_counter(b->k_base_dev, n, st);
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(st, &cs);
  if (cs == cudaStreamCaptureStatusNone) b->consumed = k;     // a captured call has not run: replays advance with lloid_graph_advance
  return LLOID_OK;
}

}  // namespace

extern "C" {

int lloid_graph_safe(const lloid_bank_t* b, int64_t n)
{
  if (!b || !b->finalized || n <= 0) return 0;
  const int64_t W = b->cfg.peak_window;
  // every replay must make the same host-side decisions as the captured call: chunk boundaries, window counts and granule
  // alignment depend on the running sample count modulo the peak window only
  return (n % W == 0 && b->consumed % W == 0 && n % b->d_max == 0) ? 1 : 0;
}

int lloid_graph_advance(lloid_bank_t* b, int64_t n)
{
  if (!b || !b->finalized) return fail(LLOID_ESTATE, "graph_advance before finalize");
  if (!lloid_graph_safe(b, n)) return fail(LLOID_EINVAL, "graph replay needs n_samples and the running sample count to be multiples of the peak window");
  b->consumed += n;
  for (lloid_bank* c : b->parts) c->consumed += n;
  return LLOID_OK;
}

int lloid_filter_host(lloid_bank_t* b, const float* strain_host, int64_t n, lloid_trigger_t* trig_host,
                      int64_t capacity, int64_t* count_host, void* stream)
{
  if (!b) return fail(LLOID_EINVAL, "null bank");
  if (!b->finalized) return fail(LLOID_ESTATE, "filter before finalize");
  if (!strain_host || !count_host || (capacity > 0 && !trig_host)) return fail(LLOID_EINVAL, "null buffer");
  if (n <= 0 || capacity < 0) return fail(LLOID_EINVAL, "bad size");
  cudaStream_t st = (cudaStream_t)stream;
  CU(cudaSetDevice(b->cfg.device));
  const size_t elems = (size_t)b->cfg.n_detectors * n;
  if (elems > b->stage_strain_elems) {
    if (b->stage_strain) { cudaFree(b->stage_strain); b->bytes -= (int64_t)b->stage_strain_elems * 4; }
    cudaError_t e = cudaMalloc((void**)&b->stage_strain, elems * 4);
    if (e != cudaSuccess) { b->stage_strain = nullptr; b->stage_strain_elems = 0; return fail(LLOID_ENOMEM, "staging alloc failed"); }
    b->stage_strain_elems = elems; b->bytes += (int64_t)elems * 4;
  }
  if (capacity > b->stage_trig_cap) {
    if (b->stage_trig) { cudaFree(b->stage_trig); b->bytes -= b->stage_trig_cap * 32; }
    cudaError_t e = cudaMalloc((void**)&b->stage_trig, (size_t)capacity * sizeof(lloid_trigger_t));
    if (e != cudaSuccess) { b->stage_trig = nullptr; b->stage_trig_cap = 0; return fail(LLOID_ENOMEM, "staging alloc failed"); }
    b->stage_trig_cap = capacity; b->bytes += capacity * 32;
  }
  CU(cudaMemcpyAsync(b->stage_strain, strain_host, elems * 4, cudaMemcpyHostToDevice, st));
  int rc = lloid_filter(b, b->stage_strain, n, b->stage_trig, capacity, (int64_t*)b->stage_count, stream);
  if (rc) return rc;
  CU(cudaMemcpyAsync(count_host, b->stage_count, 8, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  const int64_t got = std::min<int64_t>(*count_host, capacity);
  if (got > 0) {
    CU(cudaMemcpyAsync(trig_host, b->stage_trig, (size_t)got * sizeof(lloid_trigger_t), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
  }
  return lloid_check_count(*count_host, capacity);
}

int lloid_reset(lloid_bank_t* b, void* stream)
{
  if (!b) return fail(LLOID_EINVAL, "null bank");
  if (!b->finalized) return fail(LLOID_ESTATE, "reset before finalize");
  cudaStream_t st = (cudaStream_t)stream;
  CU(cudaSetDevice(b->cfg.device));
  if (!b->parts.empty()) {
    for (lloid_bank* c : b->parts) { const int rc = lloid_reset(c, stream); if (rc) return rc; }
    b->consumed = 0;
    return LLOID_OK;
  }
  CU(cudaMemsetAsync(b->hist, 0, (size_t)b->cfg.n_detectors * b->H * 4, st));
  CU(cudaMemsetAsync(b->k_base_dev, 0, 8, st));
  launch_reset_state(b->state, 2 * (int64_t)b->n_bd * b->max_templates, st);
  b->consumed = 0;
  return LLOID_OK;
}

int lloid_debug_capture(lloid_bank_t* b, int32_t bin, int32_t det, int64_t k_begin, int64_t n, float* snr_dev)
{
  int rc = check_ids(b, bin, det, 0); if (rc) return rc;
  if (!b->parts.empty()) {
    if (!b->finalized) return fail(LLOID_ESTATE, "capture before finalize");
    for (lloid_bank* c : b->parts) c->cap = Capture{nullptr, 0, 0, -1, 0};
    if (!snr_dev) return LLOID_OK;
    lloid_bank* c = b->parts[b->part_of_bin[bin]];
    return lloid_debug_capture(c, bin - c->bin_base, det, k_begin, n, snr_dev);
  }
  if (!snr_dev) { b->cap = Capture{nullptr, 0, 0, -1, 0}; return LLOID_OK; }
  if (n <= 0) return fail(LLOID_EINVAL, "capture length must be positive");
  b->cap.snr = snr_dev; b->cap.k_begin = k_begin; b->cap.n = n;
  b->cap.bd = bin * b->cfg.n_detectors + det; b->cap.rows = 2 * b->bins[bin].N;
  return LLOID_OK;
}

int64_t lloid_samples_consumed(const lloid_bank_t* b) { return b ? b->consumed : -1; }
int64_t lloid_chunk_samples(const lloid_bank_t* b) { return b ? b->C : -1; }
int64_t lloid_last_launch_count(const lloid_bank_t* b) { return b ? b->last_launches : -1; }
int64_t lloid_device_bytes(const lloid_bank_t* b)
{
  if (!b) return -1;
  int64_t v = b->bytes;
  for (const lloid_bank* c : b->parts) v += c->bytes;
  return v;
}

int lloid_set_profiling(lloid_bank_t* b, int32_t enable)
{
  if (!b) return fail(LLOID_EINVAL, "null bank");
  b->prof = enable != 0; b->events_used = 0;
  for (lloid_bank* c : b->parts) { c->prof = b->prof; c->events_used = 0; }
  return LLOID_OK;
}

int lloid_last_stage_ms(lloid_bank_t* b, float* out)
{
  if (!b || !out) return fail(LLOID_EINVAL, "null argument");
  for (int i = 0; i < 6; ++i) out[i] = 0.f;
  if (!b->parts.empty()) {                         // split bank: the parts ran back to back; their stage times add up
    for (lloid_bank* c : b->parts) {
      float v[6];
      const int rc = lloid_last_stage_ms(c, v); if (rc) return rc;
      for (int i = 0; i < 6; ++i) out[i] += v[i];
    }
    return LLOID_OK;
  }
  if (!b->prof || b->events_used < 2) return fail(LLOID_ESTATE, "profiling was not enabled for the last call");
  CU(cudaEventSynchronize(b->events[b->events_used - 1]));
  for (size_t i = 1; i < b->events_used; ++i) {
    const int tag = b->event_tag[i];
    if (tag < 0) continue;
    float ms = 0.f; CU(cudaEventElapsedTime(&ms, b->events[i - 1], b->events[i]));
    out[tag] += ms;
  }
  float ms = 0.f; CU(cudaEventElapsedTime(&ms, b->events[0], b->events[b->events_used - 1]));
  out[4] = ms;
  out[2] += out[5];                               // [5] (low-rate reconstruction kernel) is a part of [2]
  return LLOID_OK;
}

#ifdef LLOID_TRACE_BUILD
int lloid_debug_trace(long long* out, int reset) { return f16_read_trace(out, reset) ? LLOID_ECUDA : LLOID_OK; }   // scratch builds only
#endif

int lloid_path_info(const lloid_bank_t* b, int32_t* out)
{
  if (!b || !out) return fail(LLOID_EINVAL, "null argument");
  if (!b->finalized) return fail(LLOID_ESTATE, "path info before finalize");
  out[0] = out[1] = out[2] = out[3] = 0;
  if (!b->parts.empty()) {                         // split bank: all parts on the tensor kernels / any with R in TMEM / sums
    out[0] = 1;
    for (const lloid_bank* c : b->parts) {
      int32_t v[4];
      const int rc = lloid_path_info(c, v); if (rc) return rc;
      out[0] &= v[0]; out[1] |= v[1]; out[2] += v[2]; out[3] += v[3];
    }
    return LLOID_OK;
  }
  if (b->f16 && b->plan16) {
    out[0] = f16_plan_tensor_recon(b->plan16) ? 1 : 0;
    out[1] = f16_plan_r_tmem(b->plan16) ? 1 : 0;
    if (const uint8_t* ex = f16_plan_excluded(b->plan16)) for (int i = 0; i < b->n_bd; ++i) out[2] += ex[i];
    else if (!out[0]) out[2] = b->n_bd;
    for (const BinHost& B : b->bins) for (const SliceHost& S : B.slices) out[3] += S.fold ? 1 : 0;
  }
  return LLOID_OK;
}

namespace {
struct CoincGeom { long long k_w0; int n_w; long long total_t; size_t prefix_bytes, dt_bytes, table_bytes; };
CoincGeom coinc_geom(const lloid_bank* b, int64_t k_begin, int64_t n_samples)
{
  CoincGeom g;
  const long long W = b->cfg.peak_window;
  g.k_w0 = k_begin / W * W;
  g.n_w = (int)((k_begin + n_samples - g.k_w0 + W - 1) / W);
  g.total_t = 0;
  for (const BinHost& B : b->bins) g.total_t += B.N;
  g.prefix_bytes = (size_t)round_up((int64_t)(b->bins.size() + 1) * 8, 256);
  g.dt_bytes = (size_t)round_up((int64_t)b->cfg.n_detectors * b->cfg.n_detectors * 4, 256);
  g.table_bytes = (size_t)g.total_t * b->cfg.n_detectors * g.n_w * sizeof(int);
  return g;
}
}  // namespace

int64_t lloid_coincidence_scratch_bytes(const lloid_bank_t* b, int64_t k_begin, int64_t n_samples)
{
  if (!b || k_begin < 0 || n_samples <= 0) return -1;
  const CoincGeom g = coinc_geom(b, k_begin, n_samples);
  return (int64_t)(g.prefix_bytes + g.dt_bytes + g.table_bytes);
}

int lloid_coincidence(const lloid_bank_t* b, const lloid_trigger_t* trig, int64_t n, int64_t k_begin, int64_t n_samples,
                      const int32_t* max_dt, void* scratch, int64_t scratch_bytes, lloid_coinc_t* pairs, int64_t capacity,
                      int64_t* n_pairs_dev, void* stream)
{
  if (!b) return fail(LLOID_EINVAL, "null bank");
  if (!b->finalized) return fail(LLOID_ESTATE, "coincidence before finalize");
  if (!max_dt || !scratch || !n_pairs_dev || (n > 0 && !trig) || (capacity > 0 && !pairs)) return fail(LLOID_EINVAL, "null buffer");
  if (n < 0 || n > 0x7fffffffLL || capacity < 0 || k_begin < 0 || n_samples <= 0) return fail(LLOID_EINVAL, "bad size");
  const int D = b->cfg.n_detectors;
  for (int a = 0; a < D; ++a)
    for (int c = a + 1; c < D; ++c)
      if (max_dt[a * D + c] < 0 || max_dt[a * D + c] > b->cfg.peak_window)
        return fail(LLOID_EINVAL, "max_dt[%d][%d] = %d outside [0, peak_window = %d]", a, c, max_dt[a * D + c], b->cfg.peak_window);
  const CoincGeom g = coinc_geom(b, k_begin, n_samples);
  if ((int64_t)(g.prefix_bytes + g.dt_bytes + g.table_bytes) > scratch_bytes)
    return fail(LLOID_EINVAL, "scratch too small: %lld bytes needed (lloid_coincidence_scratch_bytes)", (long long)(g.prefix_bytes + g.dt_bytes + g.table_bytes));
  cudaStream_t st = (cudaStream_t)stream;
  CU(cudaSetDevice(b->cfg.device));
  std::vector<long long> prefix(b->bins.size() + 1, 0);
  for (size_t i = 0; i < b->bins.size(); ++i) prefix[i + 1] = prefix[i] + b->bins[i].N;
  char* base = (char*)scratch;
  // small pageable copies: staged by the runtime before the call returns, ordered on the stream
  CU(cudaMemcpyAsync(base, prefix.data(), prefix.size() * 8, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(base + g.prefix_bytes, max_dt, (size_t)D * D * 4, cudaMemcpyHostToDevice, st));
  launch_coincidence(trig, n, (const long long*)base, (int)b->bins.size(), D, g.k_w0, b->cfg.peak_window, g.n_w,
                     (int*)(base + g.prefix_bytes + g.dt_bytes), g.table_bytes, (const int*)(base + g.prefix_bytes), pairs, capacity,
                     (unsigned long long*)n_pairs_dev, st);
  CU(cudaGetLastError());
  return LLOID_OK;
}

void lloid_destroy(lloid_bank_t* b)
{
  if (!b) return;
  cudaSetDevice(b->cfg.device);
  cudaDeviceSynchronize();
  for (lloid_bank* c : b->parts) lloid_destroy(c);  // before the parent's arrays, which they point into
  if (b->plan16) f16_plan_destroy(b->plan16);
  for (void* p : b->owned) cudaFree(p);
  if (b->stage_strain) cudaFree(b->stage_strain);
  if (b->stage_trig) cudaFree(b->stage_trig);
  for (cudaEvent_t e : b->events) cudaEventDestroy(e);
  delete b;
}

}  // extern "C"
