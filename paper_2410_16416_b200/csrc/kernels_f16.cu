// fp16 / tcgen05 path — placeholder until the tensor-core kernels land (fails loudly, never falls back).
#include "lloid_internal.h"
#include <cstdio>
namespace lloid {
struct F16Plan { int dummy; };
F16Plan* f16_plan_create(const SliceParams*, int, const BinParams*, int, int, int, char* err, int errlen)
{ snprintf(err, errlen, "fp16 path not built yet"); return nullptr; }
void f16_plan_destroy(F16Plan* p) { delete p; }
int launch_fir_f16(F16Plan*, const SliceParams*, const RateParams*, const RateParams*, int, cudaStream_t, int64_t*) { return 1; }
int launch_recon_f16(F16Plan*, const SliceParams*, const BinParams*, const float* const*, Peak*, int, int, int64_t, Capture, cudaStream_t, int64_t*) { return 1; }
}
