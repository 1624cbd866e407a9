// Host-side plan of the fp16 / tcgen05 path, shared by kernels_f16.cu (basis FIR) and
// kernels_f16_recon.cu (reconstruction + upsample + peaks).  Not part of the ABI.
#pragma once
#include "lloid_internal.h"

#include <vector>

namespace lloid {

struct F16Plan {
  // A2 basis FIR
  int fir_grid_x = 0, fir_smem = 0, fir_stages = 0;
  int chunk_cap = 0;
  // persistent FIR (fir_f16_pers_kernel): unit lists per chunk length ([0]: the full chunk, [1]: the last one used)
  bool fir_pers = false;
  int fir_n_sm = 148, fir_hk_bytes = 0, fir_stage_cap = 0, fir_pers_stages = 0, fir_pers_smem = 0;
  // unit lists per chunk length: slot 0 = the full chunk (built at finalize), slots 1..3 = the last other lengths seen
  // (tails, streaming buffers), least recently used replaced.  Host copies are PINNED, so the upload is a true async copy.
  static constexpr int kFirSlots = 4;
  int2* fir_list_pin[kFirSlots] = {nullptr, nullptr, nullptr, nullptr};
  void* fir_list_dev[kFirSlots] = {nullptr, nullptr, nullptr, nullptr};
  cudaEvent_t fir_list_ev[kFirSlots] = {nullptr, nullptr, nullptr, nullptr};   // the slot's last upload
  int fir_list_c[kFirSlots] = {-1, -1, -1, -1}, fir_list_n[kFirSlots] = {0, 0, 0, 0};
  long long fir_list_use[kFirSlots] = {0, 0, 0, 0}, fir_tick = 0;
  size_t fir_cap_units = 0;
  // A3-A5 on the tensor cores: low-rate reconstruction (lowrate_pair_kernel) + f0-rate kernel (f0_pair_kernel)
  bool tensor_recon = false;            // false: bank outside the kernels' limits -> CUDA-core fallback
  bool r_tmem = false;                  // reconstruction kernels keep the unit's stationary R in TMEM (K <= 512) instead of shared memory
  std::vector<uint8_t> excluded;        // per (bin, detector): 1 = outside the limits, reconstructed by the FFMA kernels
  bool any_excluded = false;
  int n_bd = 0, n_lr = 0, n_sm = 148;
  int low_smem = 0, low_stages = 0, low_units = 0;
  int f0_smem = 0, f0_stages = 0, f0_ystage = 0, low_ystage = 0;   // ystage: bytes of a y ring slot per CTA
  int f0_n_pb = 0;                      // f0 schedule: template blocks per (bin, detector) when all agree (else 0)
  void* (*q_alloc)(void*, size_t) = nullptr;   // optional allocator of the rho^(d) buffers (zeroed memory or null)
  void* q_ctx = nullptr;
  int ycap = 8;                         // MMAs per y stage at most (K = 16 each)
  PairMma tab[kPairTabMax];             // interpolation MMA table of the f0 kernel (kernel parameter)
  int n_tab = 0;
  int p_bytes = 0, q_bytes = 0, l_sum_f0_max = 0, l_sum_low_max = 0;   // per CTA: band-matrix blob, rho^(d) window buffers
  PairRate rate[kNLowRates];
  std::vector<RateGroup> groups_host;   // [n_bd][n_lr]
  std::vector<BdPlan> bd_host;          // [n_bd]
  std::vector<F0Combo> combos_host;     // every (bd, template block)
  RateGroup* groups_dev = nullptr;
  BdPlan* bd_dev = nullptr;
  F0Combo* combos_dev = nullptr;
  __half* p_dev = nullptr;
  void* units_dev = nullptr;            // LowUnit[low_units], rate-major
  int units_per_rate[kNLowRates] = {0, 0, 0, 0, 0};
  SchedBd* low_cells_dev = nullptr;     // low-rate schedule: per rate class one entry per group (first unit, template blocks, cost per tile)
  int low_cells_per_rate[kNLowRates] = {0, 0, 0, 0, 0};
  SchedBd* f0_sched_dev = nullptr;      // [f0_n_bds]    f0 kernel schedule entries
  int f0_n_bds = 0;
  long long low_wsum[kNLowRates] = {0, 0, 0, 0, 0};
  long long f0_wsum = 0;
  std::vector<void*> owned;
};

// kernels_f16_recon.cu: fills the reconstruction part of the plan (returns false + err on a CUDA failure;
// an unsupported bank is not an error: tensor_recon stays false).
bool f16_plan_build_recon(F16Plan* pl, const SliceParams* sp_host, int n_problems, const BinParams* bp_host,
                          int n_bd, int chunk_cap, const double* const* up_w, int64_t* bytes, char* err, int errlen);

}  // namespace lloid
