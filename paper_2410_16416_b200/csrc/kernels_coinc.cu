// lloid_coincidence: the step after the trigger generator in the paper's flow ("These triggers are passed to the
// coincidence generator, which identifies coincidences between triggers detected with the same template and within the light
// travel time between detectors").  Works on the trigger list of ONE pass of lloid_filter over
// [k_begin, k_begin + n_samples): that list holds at most one trigger per (bin, detector, template, peak window), so a dense
// table indexed by that key finds a trigger's partners in the other detectors in O(1): window w - 1, w, w + 1 (max_dt <= W).
// Three launches: fill the table with -1, scatter the trigger indices, match.  Integer work: results are exact.
#include "../../include/lloid.h"
#include "lloid_internal.h"

namespace lloid {

__global__ void coinc_scatter_kernel(const lloid_trigger_t* __restrict__ trig, long long n, const long long* __restrict__ tmpl_off, int n_bins,
                                     int n_det, long long k_w0, int W, int n_w, int* __restrict__ table)
{
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const lloid_trigger_t t = trig[i];
  if (t.bin < 0 || t.bin >= n_bins || t.detector < 0 || t.detector >= n_det) return;
  const long long n_t = tmpl_off[t.bin + 1] - tmpl_off[t.bin];
  const long long w = (t.sample - k_w0) / W;
  if (t.template_idx < 0 || t.template_idx >= n_t || t.sample < k_w0 || w >= n_w) return;     // not a trigger of this pass: ignored
  table[((tmpl_off[t.bin] + t.template_idx) * n_det + t.detector) * n_w + w] = (int)i;
}

__global__ void coinc_match_kernel(const lloid_trigger_t* __restrict__ trig, long long n, const long long* __restrict__ tmpl_off, int n_bins,
                                   int n_det, long long k_w0, int W, int n_w, const int* __restrict__ table, const int* __restrict__ max_dt,
                                   lloid_coinc_t* __restrict__ out, long long capacity, unsigned long long* __restrict__ count)
{
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const lloid_trigger_t t = trig[i];
  if (t.bin < 0 || t.bin >= n_bins || t.detector < 0 || t.detector >= n_det) return;
  const long long n_t = tmpl_off[t.bin + 1] - tmpl_off[t.bin];
  const long long w = (t.sample - k_w0) / W;
  if (t.template_idx < 0 || t.template_idx >= n_t || t.sample < k_w0 || w >= n_w) return;
  const long long row = (tmpl_off[t.bin] + t.template_idx) * n_det;
  if (table[(row + t.detector) * n_w + w] != (int)i) return;          // a duplicate key that lost the scatter: not part of the pass
  for (int b = t.detector + 1; b < n_det; ++b) {                      // each pair once: this trigger is the lower-numbered detector's
    const int dt = max_dt[t.detector * n_det + b];
    for (long long wo = (w > 0 ? w - 1 : 0); wo <= w + 1 && wo < n_w; ++wo) {
      const int j = table[(row + b) * n_w + wo];
      if (j < 0) continue;
      long long dk = trig[j].sample - t.sample;
      if (dk < 0) dk = -dk;
      if (dk <= dt) {
        const unsigned long long slot = atomicAdd(count, 1ull);
        if ((long long)slot < capacity) { lloid_coinc_t c; c.a = i; c.b = j; out[slot] = c; }
      }
    }
  }
}

void launch_coincidence(const lloid_trigger_t* trig, long long n, const long long* tmpl_off_dev, int n_bins, int n_det, long long k_w0, int W,
                        int n_w, int* table, size_t table_bytes, const int* max_dt_dev, lloid_coinc_t* out, long long capacity,
                        unsigned long long* count, cudaStream_t st)
{
  cudaMemsetAsync(table, 0xff, table_bytes, st);
  cudaMemsetAsync(count, 0, 8, st);
  if (n <= 0) return;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  coinc_scatter_kernel<<<blocks, 256, 0, st>>>(trig, n, tmpl_off_dev, n_bins, n_det, k_w0, W, n_w, table);
  coinc_match_kernel<<<blocks, 256, 0, st>>>(trig, n, tmpl_off_dev, n_bins, n_det, k_w0, W, n_w, table, max_dt_dev, out, capacity, count);
}

}  // namespace lloid
