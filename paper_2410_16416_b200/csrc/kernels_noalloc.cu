// lloid_window_peaks_noalloc: steps A5 + A6 (|rho|^2, windowed first maximum, threshold, compaction; "identifies
// peaks in the SNR time series with SNR > 4") on a dense SNR series the CALLER holds in device memory, for callers that
// may not allocate: code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  It is the two-pass
// scheme of the bank path (one partial peak per template and 128-sample tile, then a merge per peak window) with the
// partial peaks -- which the bank path keeps in a buffer allocated at finalize -- in a FILE-SCOPE device array of a fixed
// size.  The entry point calls no cudaMalloc / cudaFree and no allocating library routine; it enqueues one 8-byte memset
// and two kernels on the caller's stream.
//
// The array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to start at zero:
// pass 1 writes every record that pass 2 of the same call reads; the one thing that must start at zero, the caller's
// trigger count, is cleared on the stream first.  Two calls that overlap on the GPU (different streams, or graph
// branches without a dependency) RACE on the array: serialise them.
#include "../../include/lloid.h"
#include "lloid_internal.h"

#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace lloid { void set_last_error(const char* msg); }

using namespace lloid;

namespace {

constexpr long long kNoAllocMaxRecords = 1ll << 19;        // 16-byte records: 8 MiB per GPU that loads the library, until exit
constexpr int kNoAllocMaxDevices = 64;

static __device__ __align__(256) Peak g_noalloc_partials[kNoAllocMaxRecords];

// In HOST code the name g_noalloc_partials is a host-side stand-in, not a device address: the kernels get the address
// cudaGetSymbolAddress returns, looked up once per device with that device current.
std::mutex g_mu;
Peak* g_scratch[kNoAllocMaxDevices];

int noalloc_fail(int code, const char* fmt, ...)
{
  char buf[512];
  va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
  set_last_error(buf);
  return code;
}

int scratch_for_current_device(Peak** out)
{
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return noalloc_fail(LLOID_ECUDA, "cudaGetDevice failed: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kNoAllocMaxDevices) return noalloc_fail(LLOID_ECUDA, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch[dev]) {
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return noalloc_fail(LLOID_ECUDA, "cudaGetDeviceProperties failed: %s", cudaGetErrorString(e));
    if (prop.major != 10) return noalloc_fail(LLOID_ECUDA, "device %d is sm_%d%d; this build is sm_100a only", dev, prop.major, prop.minor);
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_partials);
    if (e != cudaSuccess || !p) return noalloc_fail(LLOID_ECUDA, "cudaGetSymbolAddress(g_noalloc_partials) failed: %s", cudaGetErrorString(e));
    g_scratch[dev] = static_cast<Peak*>(p);
  }
  *out = g_scratch[dev];
  return LLOID_OK;
}

// pass 1: one warp per (template, 128-sample tile).  Lane l holds samples 4 l .. 4 l + 3 of the cosine and the sine row.
// First maximum: the lowest sample index wins a tie (reading R8); a NaN never wins (q > best is false).
__global__ void __launch_bounds__(256)
tile_peaks_noalloc_kernel(const float* __restrict__ snr, long long row_stride, int n_templates, int n_tiles, Peak* __restrict__ partials)
{
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int p = blockIdx.y * 8 + warp, t = blockIdx.x;
  if (p >= n_templates) return;                             // whole warps leave together
  const float4 c = __ldg(reinterpret_cast<const float4*>(snr + (size_t)(2 * p) * row_stride + (size_t)t * kTimeTile) + lane);
  const float4 s = __ldg(reinterpret_cast<const float4*>(snr + (size_t)(2 * p + 1) * row_stride + (size_t)t * kTimeTile) + lane);
  const float re4[4] = {c.x, c.y, c.z, c.w}, im4[4] = {s.x, s.y, s.z, s.w};
  float bq = -1.f, bre = 0.f, bim = 0.f;
  int bk = 4 * lane;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const float q = fmaf(re4[j], re4[j], im4[j] * im4[j]);
    if (q > bq) { bq = q; bre = re4[j]; bim = im4[j]; bk = 4 * lane + j; }
  }
#pragma unroll
  for (int x = 16; x >= 1; x >>= 1) {
    const float oq = __shfl_xor_sync(0xffffffffu, bq, x), ore = __shfl_xor_sync(0xffffffffu, bre, x), oim = __shfl_xor_sync(0xffffffffu, bim, x);
    const int ok = __shfl_xor_sync(0xffffffffu, bk, x);
    if (oq > bq || (oq == bq && ok < bk)) { bq = oq; bre = ore; bim = oim; bk = ok; }
  }
  if (lane == 0) {
    Peak pk; pk.q = bq; pk.kappa = t * kTimeTile + bk; pk.re = bre; pk.im = bim;
    partials[(size_t)t * n_templates + p] = pk;
  }
}

// pass 2: one thread per (template, complete peak window): the window's tiles in time order (a later tile wins only
// with a strictly larger |rho|^2), strict threshold, append.
__global__ void __launch_bounds__(128)
merge_noalloc_kernel(const Peak* __restrict__ partials, int n_templates, long long k_begin, long long w_first, int n_windows, int W, float theta,
                     int bin, int detector, lloid_trigger_t* __restrict__ trig, long long capacity, unsigned long long* __restrict__ count)
{
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  const int wi = blockIdx.y;
  if (p >= n_templates || wi >= n_windows) return;
  const long long w = w_first + wi;
  const int t_lo = (int)((w * W - k_begin) / kTimeTile), gt = W / kTimeTile;
  float bq = -1.f, bre = 0.f, bim = 0.f;
  int bk = -1;
  const Peak* __restrict__ pp = partials + (size_t)t_lo * n_templates + p;
  for (int g = 0; g < gt; ++g, pp += n_templates) {
    const float4 v = *reinterpret_cast<const float4*>(pp);               // Peak = {q, kappa, re, im}
    if (v.x > bq) { bq = v.x; bk = __float_as_int(v.y); bre = v.z; bim = v.w; }
  }
  if (bq >= 0.f && sqrtf(bq) > theta) {
    const unsigned long long idx = atomicAdd(count, 1ull);
    if ((long long)idx < capacity) {
      lloid_trigger_t tr;
      tr.bin = bin; tr.detector = detector; tr.template_idx = p; tr.reserved = 0;
      tr.sample = k_begin + bk; tr.snr_re = bre; tr.snr_im = bim;
      trig[idx] = tr;
    }
  }
}

}  // namespace

extern "C" {

int64_t lloid_noalloc_max_records(void) { return kNoAllocMaxRecords; }

int lloid_noalloc_setup(void)
{
  Peak* p = nullptr;
  return scratch_for_current_device(&p);
}

int lloid_window_peaks_noalloc(const float* snr_dev, int32_t n_templates, int64_t n_samples, int64_t row_stride, int64_t k_begin,
                               int32_t peak_window, float snr_threshold, int32_t bin, int32_t detector,
                               lloid_trigger_t* triggers_dev, int64_t capacity, int64_t* n_triggers_dev, void* cuda_stream)
{
  if (!snr_dev || !n_triggers_dev || (capacity > 0 && !triggers_dev)) return noalloc_fail(LLOID_EINVAL, "null buffer");
  if (n_templates < 1 || n_templates > 65536) return noalloc_fail(LLOID_EINVAL, "n_templates must be in [1, 65536]");
  if (n_samples < kTimeTile || n_samples % kTimeTile) return noalloc_fail(LLOID_EINVAL, "n_samples must be a positive multiple of %d", kTimeTile);
  if (k_begin < 0 || k_begin % kTimeTile) return noalloc_fail(LLOID_EINVAL, "k_begin must be a non-negative multiple of %d", kTimeTile);
  if (row_stride < n_samples || row_stride % 4) return noalloc_fail(LLOID_EINVAL, "row_stride must be >= n_samples and a multiple of 4 floats");
  if (reinterpret_cast<uintptr_t>(snr_dev) % 16) return noalloc_fail(LLOID_EINVAL, "snr_dev must be 16-byte aligned");
  if (peak_window < kTimeTile || peak_window % kTimeTile) return noalloc_fail(LLOID_EINVAL, "peak_window must be a positive multiple of %d", kTimeTile);
  if (!(snr_threshold >= 0.f)) return noalloc_fail(LLOID_EINVAL, "snr_threshold must be >= 0");
  if (capacity < 0) return noalloc_fail(LLOID_EINVAL, "negative capacity");
  const long long n_tiles = n_samples / kTimeTile;
  if (n_tiles > 65535 || (long long)n_templates * n_tiles > kNoAllocMaxRecords)
    return noalloc_fail(LLOID_EINVAL, "n_templates x n_samples / %d = %lld partial peaks exceed the static scratch array of %lld records (%lld MiB): "
                        "split the call in time (at peak-window boundaries) or over templates",
                        kTimeTile, (long long)n_templates * n_tiles, kNoAllocMaxRecords, kNoAllocMaxRecords * (long long)sizeof(Peak) >> 20);
  Peak* scratch = nullptr;
  if (int rc = scratch_for_current_device(&scratch)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaMemsetAsync(n_triggers_dev, 0, 8, st);             // the one value that must start at zero
  if (e != cudaSuccess) return noalloc_fail(LLOID_ECUDA, "cudaMemsetAsync failed: %s", cudaGetErrorString(e));
  dim3 g1((unsigned)n_tiles, (unsigned)((n_templates + 7) / 8));
  tile_peaks_noalloc_kernel<<<g1, 256, 0, st>>>(snr_dev, (long long)row_stride, n_templates, (int)n_tiles, scratch);
  const long long W = peak_window;
  const long long w_first = (k_begin + W - 1) / W, w_end = (k_begin + n_samples) / W;       // complete windows [w_first, w_end)
  if (w_end > w_first) {
    if (w_end - w_first > 65535) return noalloc_fail(LLOID_EINVAL, "too many peak windows in one call");
    dim3 g2((unsigned)((n_templates + 127) / 128), (unsigned)(w_end - w_first));
    merge_noalloc_kernel<<<g2, 128, 0, st>>>(scratch, n_templates, (long long)k_begin, w_first, (int)(w_end - w_first), peak_window, snr_threshold,
                                             bin, detector, triggers_dev, (long long)capacity, (unsigned long long*)n_triggers_dev);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return noalloc_fail(LLOID_ECUDA, "kernel launch failed: %s", cudaGetErrorString(e));
  return LLOID_OK;
}

}  // extern "C"
