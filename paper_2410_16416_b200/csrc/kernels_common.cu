// A1 polyphase resampler, A5/A6 peak merge + trigger compaction, state reset.
// Shared by the fp32 and fp16 paths.  See lloid_internal.h for the chunk-local coordinates.
#include "lloid_internal.h"
#include <algorithm>
#include "../../include/lloid.h"

namespace lloid {

// ------------------------------------------------------------------------------------------------
// A1  x^s[j] = sqrt(d) sum_n lp[n] x[d j - n]          (include/lloid.h A1; "downsamples")
//
// One CTA produces 256 consecutive outputs of one (rate, detector).  The strain segment it needs,
// d*256 + 2 K d samples, is read once with coalesced loads and stored de-interleaved by decimation
// phase, xsm[phi][m] = x[d (jj0 - K + m) + phi], so that in the tap loop thread t reads xsm[phi][t + a]:
// consecutive threads touch consecutive banks (a stride-d access would be a d-way bank conflict).
// Taps are pre-scaled by sqrt(d); tap index u = d a + phi.  Output in fp32 and, for the fp16 path, fp16.
// ------------------------------------------------------------------------------------------------
constexpr int kResBlock = 256;

__global__ void __launch_bounds__(kResBlock)
resample_kernel(const RateParams* __restrict__ rates, const float* __restrict__ xw, int xw_pitch,
                int xw_valid, int k_dn, int c, int want_f16)
{
  const RateParams R = rates[blockIdx.z];
  const int det = blockIdx.y;
  const int d = R.d;
  const int jj_lo = R.jj_lo_fixed;
  const int jj_hi = R.jj_hi_off + c / d;
  const int jj0 = jj_lo + blockIdx.x * kResBlock;
  if (jj0 >= jj_hi) return;
  const float* x = xw + (size_t)det * xw_pitch;
  const int t = threadIdx.x;

  if (d == 1) {                                   // fp16 copy of the full-rate stream (fp16 path only)
    const int jj = jj0 + t;
    if (want_f16 && jj < jj_hi && jj >= 0 && jj < R.xs_len) {
      const float v = (jj < xw_valid) ? x[jj] : 0.f;
      R.xs16[(size_t)det * R.xs_len + jj] = __float2half_rn(v);
    }
    return;
  }

  extern __shared__ float xsm[];
  const int mlen = kResBlock + 2 * k_dn + 1;       // odd row stride: conflict-free transposed stores
  const int seg = d * (kResBlock + 2 * k_dn) + 1;
  const int base = d * (jj0 - k_dn);               // xw index of segment element 0
  for (int i = t; i < seg; i += kResBlock) {
    const int gi = base + i;
    const float v = (gi >= 0 && gi < xw_valid) ? x[gi] : 0.f;
    xsm[(i % d) * mlen + (i / d)] = v;
  }
  __syncthreads();

  const float* __restrict__ taps = R.taps;
  float acc = 0.f;
  for (int a = 0; a < 2 * k_dn; ++a) {
    const float* tp = taps + a * d;
    for (int phi = 0; phi < d; ++phi)
      acc = fmaf(__ldg(tp + phi), xsm[phi * mlen + t + a], acc);
  }
  acc = fmaf(__ldg(taps + 2 * k_dn * d), xsm[t + 2 * k_dn], acc);   // last tap: a = 2K, phi = 0

  const int jj = jj0 + t;
  if (jj < jj_hi && jj >= 0 && jj < R.xs_len) {
    const size_t o = (size_t)det * R.xs_len + jj;
    R.xs32[o] = acc;
    if (want_f16) R.xs16[o] = __float2half_rn(acc);
  }
}

// Register-tiled variant (K_dn even): one thread produces 4 consecutive outputs with a sliding window of the
// strain in registers, so one shared-memory load and one (broadcast) tap load feed 4 FMAs.  The segment is stored
// xs4[phi][m & 3][m >> 2] (decimation phase, then the residue of the low-rate index): thread t reads quotient
// t + const of one residue row -- consecutive banks -- for every window element.  Taps are staged per phase,
// tp[phi][a] = taps[a d + phi].  128 threads x 4 = 512 outputs per CTA.
constexpr int kRes4Threads = 128, kRes4Out = 4 * kRes4Threads;

__global__ void __launch_bounds__(kRes4Threads)
resample4_kernel(const RateParams* __restrict__ rates, int rate_base, const float* __restrict__ xw, int xw_pitch,
                 int xw_valid, int k_dn, int c, int want_f16)
{
  // rates are stored by ascending d and a CTA's work grows with d: the largest d of the launch is dispatched first (short tail)
  const RateParams R = rates[rate_base + gridDim.z - 1 - blockIdx.z];
  const int det = blockIdx.y;
  const int d = R.d;
  const int jj_lo = R.jj_lo_fixed;
  const int jj_hi = R.jj_hi_off + c / d;
  const int jj0 = jj_lo + blockIdx.x * kRes4Out;
  if (jj0 >= jj_hi) return;
  const float* x = xw + (size_t)det * xw_pitch;
  const int t = threadIdx.x;

  if (d == 1) {                                   // fp16 copy of the full-rate stream (fp16 path only)
    if (want_f16)
      for (int i = t; i < kRes4Out; i += kRes4Threads) {
        const int jj = jj0 + i;
        if (jj < jj_hi && jj >= 0 && jj < R.xs_len) R.xs16[(size_t)det * R.xs_len + jj] = __float2half_rn(jj < xw_valid ? x[jj] : 0.f);
      }
    return;
  }

  extern __shared__ float xsm[];
  const int K2 = 2 * k_dn;
  const int Q = (kRes4Out + K2) / 4 + 1;          // quotients per residue row
  float* xs4 = xsm;                               // [d][4][Q]
  float* tp = xsm + (size_t)d * 4 * Q;            // [d][K2], then the last tap
  const int seg = d * (kRes4Out + K2) + 1;
  const int base = d * (jj0 - k_dn);              // xw index of segment element 0
  const int l2d = 31 - __clz(d);
  for (int i = t; i < seg; i += kRes4Threads) {
    const int gi = base + i;
    const float v = (gi >= 0 && gi < xw_valid) ? x[gi] : 0.f;
    const int m = i >> l2d, phi = i & (d - 1);     // d is a power of two: the division cost as much as the filter itself
    xs4[(phi * 4 + (m & 3)) * Q + (m >> 2)] = v;
  }
  for (int i = t; i < K2 * d + 1; i += kRes4Threads) {
    const int a = i >> l2d, phi = i & (d - 1);
    tp[(a == K2) ? d * K2 : phi * K2 + a] = __ldg(R.taps + i);
  }
  __syncthreads();

  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
  for (int phi = 0; phi < d; ++phi) {
    const float* __restrict__ xb = xs4 + (size_t)phi * 4 * Q + t;
    const float* __restrict__ tb = tp + phi * K2;
    float w0 = xb[0], w1 = xb[Q], w2 = xb[2 * Q], w3 = xb[3 * Q];
#pragma unroll 4
    for (int a4 = 0; a4 < K2; a4 += 4) {
      const int qn = (a4 >> 2) + 1;
      const float4 tv = *reinterpret_cast<const float4*>(tb + a4);
      const float n0 = xb[qn], n1 = xb[Q + qn], n2 = xb[2 * Q + qn], n3 = xb[3 * Q + qn];
      a0 = fmaf(tv.x, w0, a0); a1 = fmaf(tv.x, w1, a1); a2 = fmaf(tv.x, w2, a2); a3 = fmaf(tv.x, w3, a3);
      a0 = fmaf(tv.y, w1, a0); a1 = fmaf(tv.y, w2, a1); a2 = fmaf(tv.y, w3, a2); a3 = fmaf(tv.y, n0, a3);
      a0 = fmaf(tv.z, w2, a0); a1 = fmaf(tv.z, w3, a1); a2 = fmaf(tv.z, n0, a2); a3 = fmaf(tv.z, n1, a3);
      a0 = fmaf(tv.w, w3, a0); a1 = fmaf(tv.w, n0, a1); a2 = fmaf(tv.w, n1, a2); a3 = fmaf(tv.w, n2, a3);
      w0 = n0; w1 = n1; w2 = n2; w3 = n3;
    }
  }
  {                                               // last tap: a = 2K, phi = 0; after the loop w_i = x[m = 4t + i + 2K] of phase d-1,
    const float tl = tp[d * K2];                  // so re-read phase 0
    const float* __restrict__ xb = xs4 + t + (K2 >> 2);
    a0 = fmaf(tl, xb[0], a0); a1 = fmaf(tl, xb[Q], a1); a2 = fmaf(tl, xb[2 * Q], a2); a3 = fmaf(tl, xb[3 * Q], a3);
  }
  const float acc[4] = {a0, a1, a2, a3};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int jj = jj0 + 4 * t + i;
    if (jj < jj_hi && jj >= 0 && jj < R.xs_len) {
      const size_t o = (size_t)det * R.xs_len + jj;
      R.xs32[o] = acc[i];
      if (want_f16) R.xs16[o] = __float2half_rn(acc[i]);
    }
  }
}

int configure_common_kernels()              // per device, at finalize (see configure_f32_kernels)
{
  cudaError_t e = set_max_dyn_smem(resample_kernel);
  if (e == cudaSuccess) e = set_max_dyn_smem(resample4_kernel);
  return e == cudaSuccess ? 0 : 1;
}

void launch_resample(const RateParams* rates_dev, const RateParams* rates_host, int n_rates,
                     const float* xw, int xw_pitch, int xw_valid, int n_det, int k_dn, int c,
                     bool want_f16, cudaStream_t st, int64_t* launches)
{
  int max_blocks = 0, max_d = 1;
  bool any = false;
  for (int r = 0; r < n_rates; ++r) {
    const RateParams& R = rates_host[r];
    if (R.d == 1 && !want_f16) continue;
    any = true;
    const int span = R.jj_hi_off + c / R.d - R.jj_lo_fixed;
    const int nb = (span + kResBlock - 1) / kResBlock;
    if (nb > max_blocks) max_blocks = nb;
    if (R.d > max_d) max_d = R.d;
  }
  if (!any || max_blocks <= 0) return;
  const size_t smem = sizeof(float) * (size_t)max_d * (kResBlock + 2 * k_dn + 1);

  if (k_dn % 2 == 0) {                              // register-tiled kernel: 512 outputs per CTA
    // Two launches, d <= 8 and d >= 16 (rates are sorted by d): the shared-memory segment of a CTA grows with d (75 KB at
    // d = 32, three CTAs per SM), and in ONE launch sized for the largest d the many small-d CTAs ran at three per SM too
    // (ncu: 17 % of the warp slots, FMA pipe 17 %).  0.75 -> 0.47 ms per config-2 step; one launch per d was slower again.
    const int Q = (kRes4Out + 2 * k_dn) / 4 + 1;
    int r0 = 0;
    while (r0 < n_rates) {
      int r1 = r0, gmax_d = 1, blocks4 = 0;
      const bool one = c <= 16384;                 // short buffers (streaming): a second launch costs more than it saves
      const bool small = one || rates_host[r0].d <= 8;
      while (r1 < n_rates && (one || rates_host[r1].d <= 8) == small) {
        const RateParams& R = rates_host[r1];
        if (!(R.d == 1 && !want_f16)) {
          const int span = R.jj_hi_off + c / R.d - R.jj_lo_fixed;
          blocks4 = std::max(blocks4, (span + kRes4Out - 1) / kRes4Out);
          gmax_d = std::max(gmax_d, R.d);
        }
        ++r1;
      }
      if (blocks4 > 0) {
        const size_t smem4 = sizeof(float) * ((size_t)gmax_d * 4 * Q + (size_t)gmax_d * 2 * k_dn + 4);
        dim3 grid4(blocks4, n_det, r1 - r0);
        resample4_kernel<<<grid4, kRes4Threads, smem4, st>>>(rates_dev, r0, xw, xw_pitch, xw_valid, k_dn, c, want_f16 ? 1 : 0);
        ++*launches;
      }
      r0 = r1;
    }
    return;
  }
  dim3 grid(max_blocks, n_det, n_rates);
  resample_kernel<<<grid, kResBlock, smem, st>>>(rates_dev, xw, xw_pitch, xw_valid, k_dn, c, want_f16 ? 1 : 0);
  ++*launches;
}

// ------------------------------------------------------------------------------------------------
// A5/A6  merge the per-tile partial maxima into the maximum of every peak window [wW, (w+1)W) the chunk
// touches, emit a trigger for every window the chunk completes with |rho| > theta (strict),
// and carry the maximum of an unfinished last window to the next chunk / call (A8).
// One thread per (bin, detector, template, window touched by the chunk); tiles are visited in time order
// so that the first (lowest k) maximum wins ties (R8).  Chunk starts and W are multiples of the
// tile length, so a tile never straddles two windows.  The carried state is double-buffered (state_in is
// the previous chunk's state_out): the thread of the first window reads it, the thread of the last one
// writes it, and they are different threads whenever the chunk touches more than one window.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
merge_windows_kernel(const BinParams* __restrict__ bp, int max_templates, const Peak* __restrict__ partials,
                     int slots_cap, const int32_t* __restrict__ slot_tiles, int c, const long long* __restrict__ k_base, long long k_off,
                     int W, float theta,
                     const PeakState* __restrict__ state_in, PeakState* __restrict__ state_out, int n_det, int bin_base,
                     lloid_trigger_t* __restrict__ trig, long long capacity, unsigned long long* __restrict__ count)
{
  const int bd = blockIdx.y;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  const BinParams B = bp[bd];
  if (p >= B.n_templates) return;
  // absolute index of the chunk's first sample: the call's first sample is read from DEVICE memory (advanced on the stream at
  // the end of every lloid_filter call), so a call captured in a CUDA graph stamps the right times when it is replayed
  const long long k_a = *k_base + k_off;
  const long long w_first = k_a / W, w_last = (k_a + c - 1) / W;
  const long long w = w_first + blockIdx.z;
  if (w > w_last) return;
  const long long lo = (w * W > k_a) ? w * W : k_a;
  const long long hi = ((w + 1) * W < k_a + c) ? (w + 1) * W : k_a + c;
  PeakState s;
  if (w * W < k_a) s = state_in[(size_t)bd * max_templates + p];      // window began in an earlier chunk
  else { s.q = -1.f; s.re = 0.f; s.im = 0.f; s.pad = 0; s.k = -1; }
  // partial slots: runs of gt tiles aligned to absolute multiples of gt tiles (gt = 1: one slot per tile), n_rec records per
  // run (the tensor f0 kernel's two epilogue groups write one each: slot_tiles = gt | 1 << 16).  Records of a run are not
  // in time order: the larger |rho|^2 wins, the earlier sample on a tie (R8).
  const int st = slot_tiles ? slot_tiles[bd] : 1;
  const int gt = st & 0xffff, n_rec = (st >> 16) ? 2 : 1;
  const long long a0 = k_a / kTimeTile;
  const int t_lo = (int)((lo - k_a) / kTimeTile), t_hi = (int)((hi - k_a + kTimeTile - 1) / kTimeTile);   // tiles [t_lo, t_hi)
  const int g0 = n_rec * (int)((a0 + t_lo) / gt - a0 / gt), g1 = n_rec * ((int)((a0 + t_hi - 1) / gt - a0 / gt) + 1);
  const Peak* __restrict__ pp = partials + ((size_t)bd * slots_cap + g0) * max_templates + p;
  for (int g = g0; g < g1; g += 8) {               // 8 independent 16-byte loads in flight per thread, then the ordered compare
    float4 v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
      v[i] = (g + i < g1) ? __ldcs(reinterpret_cast<const float4*>(pp + (size_t)i * max_templates)) : make_float4(-2.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < 8; ++i) {                   // Peak = {q, kappa, re, im}
      const long long k = k_a + __float_as_int(v[i].y);
      if (v[i].x > s.q || (v[i].x == s.q && k < s.k)) { s.q = v[i].x; s.re = v[i].z; s.im = v[i].w; s.k = k; }
    }
    pp += (size_t)8 * max_templates;
  }
  const bool complete = (w + 1) * W <= k_a + c;
  if (complete && s.q >= 0.f && sqrtf(s.q) > theta) {
    const unsigned long long idx = atomicAdd(count, 1ull);
    if ((long long)idx < capacity) {
      lloid_trigger_t t;
      t.bin = bin_base + bd / n_det; t.detector = bd % n_det; t.template_idx = p; t.reserved = 0;
      t.sample = s.k; t.snr_re = s.re; t.snr_im = s.im;
      trig[idx] = t;
    }
  }
  if (w == w_last) {
    if (complete) { s.q = -1.f; s.re = 0.f; s.im = 0.f; s.pad = 0; s.k = -1; }
    state_out[(size_t)bd * max_templates + p] = s;
  }
}

void launch_merge_windows(const BinParams* bp_dev, int n_bd, int max_templates, const Peak* partials,
                          int slots_cap, const int32_t* slot_tiles_dev, int c, int64_t k_a, const long long* k_base_dev, int64_t k_off,
                          int W, float theta,
                          const PeakState* state_in, PeakState* state_out, int n_det, int bin_base, void* triggers, int64_t capacity,
                          unsigned long long* count, cudaStream_t st, int64_t* launches)
{
  const int n_w = (int)((k_a + c - 1) / W - k_a / W) + 1;      // host copy of k_a: only the launch geometry depends on it
  dim3 grid((max_templates + 127) / 128, n_bd, n_w);
  merge_windows_kernel<<<grid, 128, 0, st>>>(bp_dev, max_templates, partials, slots_cap, slot_tiles_dev, c, k_base_dev, (long long)k_off, W,
                                            theta, state_in, state_out, n_det, bin_base, (lloid_trigger_t*)triggers,
                                            (long long)capacity, count);
  ++*launches;
}

__global__ void advance_counter_kernel(long long* k_base, long long n) { *k_base += n; }
void launch_advance_counter(long long* k_base_dev, int64_t n, cudaStream_t st) { advance_counter_kernel<<<1, 1, 0, st>>>(k_base_dev, (long long)n); }

__global__ void reset_state_kernel(PeakState* s, long long n)
{
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { PeakState e; e.q = -1.f; e.re = 0.f; e.im = 0.f; e.pad = 0; e.k = -1; s[i] = e; }
}

void launch_reset_state(PeakState* state, int64_t n, cudaStream_t st)
{
  if (n <= 0) return;
  reset_state_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(state, (long long)n);
}

}  // namespace lloid
