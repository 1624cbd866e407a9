// fp16 path (LLOID_F16): A2 basis FIR on the tcgen05 tensor cores.
//
//   y^s_l[j] = sum_t U^s[l,t] x^s[j - n_s + t]                 (include/lloid.h A2)
//
// As a GEMM:  Y[time j, l] = H[j, t] * U[l, t]^T  with the Hankel matrix H[j, t] = x^s[b0 + j + t].
// H is never materialised.  In the no-swizzle K-major operand layout a core matrix is 8 rows x 8 fp16
// (128 contiguous bytes), and core matrix (row group jg, tap group tg) of a Hankel matrix depends only
// on q = jg + tg:   Cq[r][e] = x[b0 + 8 q + r + e].   So ONE array C of (rows + taps)/8 core matrices
// (16 bytes per sample of the strain window) serves as the A operand of every MMA of the tile with
// descriptor strides LBO = SBO = 128 bytes; the K loop only advances the start address.  The window is
// staged once per CTA; U streams through shared memory in pre-packed 64-tap stages (one 1-D bulk copy
// each, mbarrier pipeline); MT time tiles of 128 rows share every U stage (MT accumulators in TMEM).
//
// Warp roles (192 threads): warp 0 = bulk-copy producer, warp 1 = MMA issuer, warps 2-5 = epilogue
// (TMEM -> registers -> fp16 -> Y, packed in the Y16 layout of lloid_internal.h (64-row tiles) that the
// reconstruction kernels fetch with 1-D bulk copies as an MMA operand).
#include "f16_plan.h"
#include "tc05.cuh"

#include <algorithm>
#include <cstdio>
#include <vector>

namespace lloid {

using namespace tc;

constexpr int FH_THREADS = 192;
constexpr int FH_KB = 64;                    // taps per pipeline stage
constexpr int FH_MAX_STAGES = 8;

__host__ __device__ __forceinline__ int fir_mt(int L_pad) { int mt = 512 / L_pad; return mt > 4 ? 4 : (mt < 1 ? 1 : mt); }
static inline int fir_mt_host(int L_pad) { int mt = 512 / L_pad; return mt > 4 ? 4 : (mt < 1 ? 1 : mt); }

__global__ void __launch_bounds__(FH_THREADS, 1)
fir_f16_kernel(const SliceParams* __restrict__ sp, const RateParams* __restrict__ rates, int o, int c, int n_stages)
{
  const SliceParams P = sp[blockIdx.y];
  const int rows_needed = (c >> P.log2d) + P.fir_halo;
  const int L_pad = P.L_pad;
  const int MT = fir_mt(L_pad);
  const int r0 = blockIdx.x * 128 * MT;
  if (r0 >= rows_needed) return;
  int mt_used = (rows_needed - r0 + 127) / 128; if (mt_used > MT) mt_used = MT;

  const int n_kb = (P.n_taps + FH_KB - 1) / FH_KB;
  const int n_pad = n_kb * FH_KB;
  const int n_chunks = mt_used * 128 + n_pad;                 // 16-byte chunks of the Hankel array
  const int stage_bytes = L_pad * FH_KB * 2;

  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t bar_full[FH_MAX_STAGES], bar_empty[FH_MAX_STAGES], bar_acc;
  __shared__ uint32_t tmem_slot;
  uint8_t* sC = smem;                                          // [n_chunks][16 B]
  uint8_t* sRaw = sC + (size_t)n_chunks * 16;                  // raw fp16 window, n_chunks + 8 samples (+pad)
  uint8_t* sB = sRaw + (((size_t)(n_chunks + 16) * 2 + 127) / 128) * 128;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  if (tid == 32) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(smem_u32(&bar_full[s]), 1); mbar_init(smem_u32(&bar_empty[s]), 1); }
    mbar_init(smem_u32(&bar_acc), 1);
    mbar_init_fence();
  }

  // ---- stage the strain window and expand it into the Hankel core-matrix array --------------------
  const RateParams R = rates[P.rate_idx];
  const __half* __restrict__ xs = R.xs16 + (size_t)P.det * R.xs_len;
  const int b0 = P.jjY0 + (o >> P.log2d) + r0 - P.n_taps;       // xs index of window element 0 (>= 0)
  {
    unsigned short* raw = reinterpret_cast<unsigned short*>(sRaw);
    const unsigned short* xg = reinterpret_cast<const unsigned short*>(xs);
    for (int i = tid; i < n_chunks + 8; i += FH_THREADS) {
      const int idx = b0 + i;
      raw[i] = (idx >= 0 && idx < R.xs_len) ? __ldg(xg + idx) : (unsigned short)0;
    }
  }
  __syncthreads();
  {
    const uint32_t* raw32 = reinterpret_cast<const uint32_t*>(sRaw);
    for (int ch = tid; ch < n_chunks; ch += FH_THREADS) {      // chunk ch = window samples [ch, ch + 8)
      const int w = ch >> 1;
      uint32_t a0 = raw32[w], a1 = raw32[w + 1], a2 = raw32[w + 2], a3 = raw32[w + 3];
      if (ch & 1) {
        const uint32_t a4 = raw32[w + 4];
        a0 = __funnelshift_r(a0, a1, 16); a1 = __funnelshift_r(a1, a2, 16);
        a2 = __funnelshift_r(a2, a3, 16); a3 = __funnelshift_r(a3, a4, 16);
      }
      *reinterpret_cast<uint4*>(sC + (size_t)ch * 16) = make_uint4(a0, a1, a2, a3);
    }
  }
  fence_async_smem();                                          // generic-proxy writes -> visible to the MMA (async proxy)
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem = tmem_slot;

  if (warp == 0) {
    // ===== producer: one elected thread (ptxas keeps an elect.sync-guarded loop in uniform registers; a per-lane
    // predicate on the issuing instruction costs an R2UR waterfall per instruction): U stages, pre-packed
    // [kb][tap group 8][l L_pad][8 taps] =====
    if (elect_one()) {
    const uint8_t* src = reinterpret_cast<const uint8_t*>(P.U16);
    const int n_kb_u = n_kb;
    const uint32_t sbytes = (uint32_t)stage_bytes;
    const uint32_t bfull = smem_u32(&bar_full[0]), bempty = smem_u32(&bar_empty[0]), sB_u = smem_u32(sB);
    int s = 0; uint32_t ph = 0;
    for (int kb = 0; kb < n_kb_u; ++kb, src += sbytes) {
      mbar_wait(bempty + 8u * s, ph ^ 1u);
      mbar_expect_tx(bfull + 8u * s, sbytes);
      bulk_g2s(sB_u + (uint32_t)s * sbytes, src, sbytes, bfull + 8u * s);
      if (++s == n_stages) { s = 0; ph ^= 1u; }
    }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: one elected thread =====
    if (elect_one()) {
    const int Lp_u = L_pad, n_kb_u = n_kb, mt_u = mt_used;
    const int n_split = (Lp_u > 256) ? 2 : 1;
    const int Nmma = Lp_u / n_split;
    const uint32_t idesc = idesc_f16(128, Nmma);
    const uint32_t bfull = smem_u32(&bar_full[0]), bempty = smem_u32(&bar_empty[0]);
    const uint32_t c_lo = desc_lo(smem_u32(sC), 128u);                         // Hankel array: LBO = SBO = 128
    const uint32_t b_lo0 = desc_lo(smem_u32(sB), (uint32_t)(Lp_u * 16));
    const uint32_t b_step = (uint32_t)(Lp_u * FH_KB * 2) >> 4, b_k16 = (uint32_t)(2 * Lp_u);
    const uint32_t tm = tmem;
    int s = 0; uint32_t ph = 0;
    for (int kb = 0; kb < n_kb_u; ++kb) {
      mbar_wait(bfull + 8u * s, ph);
      fence_after();
      {
        const uint32_t b_lo = b_lo0 + (uint32_t)s * b_step;
        for (int mt = 0; mt < mt_u; ++mt) {
          const uint32_t a_lo = c_lo + (uint32_t)(mt * 16 + kb * 8) * 8u;
          const uint32_t d_t = tm + (uint32_t)(mt * Lp_u);
#pragma unroll
          for (int k16 = 0; k16 < FH_KB / 16; ++k16) {
            const uint64_t adesc = desc64(a_lo + (uint32_t)(k16 * 16));
            for (int h = 0; h < n_split; ++h)
              mma_ss(d_t + (uint32_t)(h * Nmma), adesc, desc64(b_lo + (uint32_t)k16 * b_k16 + (uint32_t)(h * Nmma)), idesc,
                       (kb | k16) ? 1u : 0u);
          }
        }
        commit(bempty + 8u * s);                                       // stage reusable once these MMAs have read it
      }
      if (++s == n_stages) { s = 0; ph ^= 1u; }
    }
    commit(smem_u32(&bar_acc));
    }
  } else {
    // ===== epilogue: TMEM -> fp16 -> Y16[lc][row][8] =====
    const int q = warp & 3;                                    // TMEM lane quarter this warp may access
    mbar_wait(smem_u32(&bar_acc), 0);
    fence_after();
    __half* __restrict__ Y = reinterpret_cast<__half*>(P.Y);
    for (int mt = 0; mt < mt_used; ++mt) {
      const int row = (r0 + mt * 128 + q * 32 + lane) * P.out_mul + P.out_add;           // folded slice: phase rows interleave
      __half* __restrict__ Yt = reinterpret_cast<__half*>(reinterpret_cast<char*>(Y) + (size_t)(row >> 6) * P.y_step64) + (row & 63) * 8;   // Y16[64-row tile][slice][lc][row % 64][8]
      const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(mt * L_pad);
      for (int c0 = 0; c0 < L_pad; c0 += 16) {
        uint32_t v[16];
        tmem_ld16(taddr + c0, v);
        tmem_ld_wait();
        if (row < P.y_rows_cap) {
          uint32_t h[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const __half2 p = __floats2half2_rn(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1]));
            h[i] = *reinterpret_cast<const uint32_t*>(&p);
          }
          const size_t lc = (size_t)(c0 >> 3);
          *reinterpret_cast<uint4*>(Yt + lc * 512) = make_uint4(h[0], h[1], h[2], h[3]);
          *reinterpret_cast<uint4*>(Yt + (lc + 1) * 512) = make_uint4(h[4], h[5], h[6], h[7]);
        }
      }
    }
  }
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
// Persistent variant: one CTA per SM walks the (slice problem, block of MT time tiles) units
// list[blockIdx.x], list[blockIdx.x + gridDim.x], ...: the host sorts the units by descending cost and deals them in
// serpentine order, so the SMs finish within ~5 % of each other and neighbours in the list (same slice) share U in L2.
// What the one-unit-per-CTA kernel serialises is overlapped here:
//   warps 6-9  stage the strain window of the NEXT unit and expand it into the second Hankel buffer,
//   warp 0     keeps the U ring full across unit boundaries,
//   warp 1     issues the MMAs (one elected thread),
//   warps 2-5  drain the accumulators of the previous unit (TMEM -> fp16 -> Y16); only this drain is still exposed,
//              because MT x L_pad accumulator columns leave no room for a second set.
// TMEM, the barriers and the ring are set up once per launch instead of once per unit.
constexpr int FP_THREADS = 320;

struct FirUnit {                   // what every role derives from the unit index
  int valid, p, r0, mt_used, n_kb, n_chunks, L_pad, b0;
};

__device__ __forceinline__ FirUnit fir_unit(const SliceParams* __restrict__ sp, const int2* __restrict__ list, int u, int o, int c)
{
  FirUnit U;
  const int2 e = list[u];                // (problem, block of MT time tiles), dealt to the CTAs by descending cost
  U.p = e.x;
  const SliceParams* P = sp + U.p;
  const int d = P->d, log2d = P->log2d, n_taps = P->n_taps;
  U.L_pad = P->L_pad;
  const int rows_needed = (c >> log2d) + P->fir_halo;
  const int MT = fir_mt(U.L_pad);
  U.r0 = e.y * 128 * MT;
  U.valid = U.r0 < rows_needed;
  int m = (rows_needed - U.r0 + 127) / 128; U.mt_used = m > MT ? MT : m;
  U.n_kb = (n_taps + FH_KB - 1) / FH_KB;
  U.n_chunks = U.mt_used * 128 + U.n_kb * FH_KB;
  U.b0 = P->jjY0 + (o >> log2d) + U.r0 - n_taps;
  return U;
}

__global__ void __launch_bounds__(FP_THREADS, 1)
fir_f16_pers_kernel(const SliceParams* __restrict__ sp, const RateParams* __restrict__ rates, int o, int c, int n_stages,
                    const int2* __restrict__ list, int n_units, int hk_bytes, int stage_cap)
{
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) uint64_t bar_full[FH_MAX_STAGES], bar_empty[FH_MAX_STAGES], hk_full[2], hk_empty[2], acc_full, acc_empty;
  __shared__ uint32_t tmem_slot;
  // [2] x { Hankel array (n_chunks x 16 B) | raw fp16 window }, then the U ring
  uint8_t* sB = smem + 2 * (size_t)hk_bytes;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  if (tid == 32) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(smem_u32(&bar_full[s]), 1); mbar_init(smem_u32(&bar_empty[s]), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(smem_u32(&hk_full[b]), 128); mbar_init(smem_u32(&hk_empty[b]), 1); }
    mbar_init(smem_u32(&acc_full), 1); mbar_init(smem_u32(&acc_empty), 128);
    mbar_init_fence();
  }
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t bfull = smem_u32(&bar_full[0]), bempty = smem_u32(&bar_empty[0]);

  if (warp >= 6) {
    // ===== stagers (128 threads): strain window -> raw fp16 -> Hankel core-matrix array, double-buffered =====
    const int st = tid - 192;
    int k = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const FirUnit U = fir_unit(sp, list, u, o, c);
      if (!U.valid) continue;
      const int b = k & 1;
      uint8_t* sC = smem + (size_t)b * hk_bytes;
      uint8_t* sRaw = sC + (size_t)U.n_chunks * 16;
      if (k >= 2) mbar_wait(smem_u32(&hk_empty[b]), (uint32_t)((k >> 1) - 1) & 1u);     // MMAs that read this buffer are complete
      const SliceParams* P = sp + U.p;
      const RateParams* R = rates + P->rate_idx;
      const int xs_len = R->xs_len;
      const unsigned short* xg = reinterpret_cast<const unsigned short*>(R->xs16 + (size_t)P->det * xs_len);
      unsigned short* raw = reinterpret_cast<unsigned short*>(sRaw);
      for (int i = st; i < U.n_chunks + 8; i += 128) {
        const int idx = U.b0 + i;
        raw[i] = (idx >= 0 && idx < xs_len) ? __ldg(xg + idx) : (unsigned short)0;
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");
      const uint32_t* raw32 = reinterpret_cast<const uint32_t*>(sRaw);
      for (int ch = st; ch < U.n_chunks; ch += 128) {            // chunk ch = window samples [ch, ch + 8)
        const int w = ch >> 1;
        uint32_t a0 = raw32[w], a1 = raw32[w + 1], a2 = raw32[w + 2], a3 = raw32[w + 3];
        if (ch & 1) {
          const uint32_t a4 = raw32[w + 4];
          a0 = __funnelshift_r(a0, a1, 16); a1 = __funnelshift_r(a1, a2, 16);
          a2 = __funnelshift_r(a2, a3, 16); a3 = __funnelshift_r(a3, a4, 16);
        }
        *reinterpret_cast<uint4*>(sC + (size_t)ch * 16) = make_uint4(a0, a1, a2, a3);
      }
      fence_async_smem();                                        // generic-proxy writes -> visible to the MMAs (async proxy)
      mbar_arrive(smem_u32(&hk_full[b]));
      asm volatile("bar.sync 1, 128;" ::: "memory");             // raw of this buffer may be overwritten two units later only
      ++k;
    }
  } else if (warp == 0) {
    // ===== producer: one elected thread; the U ring runs on across unit boundaries =====
    if (elect_one()) {
      const uint32_t sB_u = smem_u32(sB);
      int s = 0; uint32_t ph = 0;
      for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const FirUnit U = fir_unit(sp, list, u, o, c);
        if (!U.valid) continue;
        const uint8_t* src = reinterpret_cast<const uint8_t*>(sp[U.p].U16);
        const uint32_t sbytes = (uint32_t)(U.L_pad * FH_KB * 2);
        for (int kb = 0; kb < U.n_kb; ++kb, src += sbytes) {
          mbar_wait(bempty + 8u * s, ph ^ 1u);
          mbar_expect_tx(bfull + 8u * s, sbytes);
          bulk_g2s(sB_u + (uint32_t)s * (uint32_t)stage_cap, src, sbytes, bfull + 8u * s);
          if (++s == n_stages) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: one elected thread =====
    if (elect_one()) {
      int s = 0; uint32_t ph = 0;
      int k = 0;
      for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
        const FirUnit U = fir_unit(sp, list, u, o, c);
        if (!U.valid) continue;
        const int b = k & 1;
        const int Lp = U.L_pad;
        const int n_split = (Lp > 256) ? 2 : 1;
        const int Nmma = Lp / n_split;
        const uint32_t idesc = idesc_f16(128, Nmma);
        const uint32_t c_lo = desc_lo(smem_u32(smem + (size_t)b * hk_bytes), 128u);      // Hankel array: LBO = SBO = 128
        const uint32_t b_lo0 = desc_lo(smem_u32(sB), (uint32_t)(Lp * 16));
        const uint32_t b_step = (uint32_t)stage_cap >> 4, b_k16 = (uint32_t)(2 * Lp);
        mbar_wait(smem_u32(&hk_full[b]), (uint32_t)(k >> 1) & 1u);                       // this unit's Hankel array is built
        if (k >= 1) mbar_wait(smem_u32(&acc_empty), (uint32_t)(k - 1) & 1u);             // the previous unit's accumulators are drained
        fence_after();
        for (int kb = 0; kb < U.n_kb; ++kb) {
          mbar_wait(bfull + 8u * s, ph);
          fence_after();
          const uint32_t b_lo = b_lo0 + (uint32_t)s * b_step;
          for (int mt = 0; mt < U.mt_used; ++mt) {
            const uint32_t a_lo = c_lo + (uint32_t)(mt * 16 + kb * 8) * 8u;
            const uint32_t d_t = tmem + (uint32_t)(mt * Lp);
#pragma unroll
            for (int k16 = 0; k16 < FH_KB / 16; ++k16) {
              const uint64_t adesc = desc64(a_lo + (uint32_t)(k16 * 16));
              for (int h = 0; h < n_split; ++h)
                mma_ss(d_t + (uint32_t)(h * Nmma), adesc, desc64(b_lo + (uint32_t)k16 * b_k16 + (uint32_t)(h * Nmma)), idesc,
                       (kb | k16) ? 1u : 0u);
            }
          }
          commit(bempty + 8u * s);                                 // stage reusable once these MMAs have read it
          if (++s == n_stages) { s = 0; ph ^= 1u; }
        }
        commit(smem_u32(&hk_empty[b]));                            // Hankel buffer reusable once every MMA of the unit is complete
        commit(smem_u32(&acc_full));
        ++k;
      }
    }
  } else {
    // ===== epilogue (warps 2-5): TMEM -> fp16 -> Y16[lc][row][8] =====
    const int q = warp & 3;                                        // TMEM lane quarter this warp may access
    int k = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const FirUnit U = fir_unit(sp, list, u, o, c);
      if (!U.valid) continue;
      const SliceParams* P = sp + U.p;
      __half* __restrict__ Y = reinterpret_cast<__half*>(P->Y);
      const int y_rows_cap = P->y_rows_cap, y_step64 = P->y_step64;
      const int L_pad = U.L_pad;
        mbar_wait(smem_u32(&acc_full), (uint32_t)k & 1u);
      fence_after();
      for (int mt = 0; mt < U.mt_used; ++mt) {
        const int row = (U.r0 + mt * 128 + q * 32 + lane) * P->out_mul + P->out_add;       // folded slice: phase rows interleave
        __half* __restrict__ Yt = reinterpret_cast<__half*>(reinterpret_cast<char*>(Y) + (size_t)(row >> 6) * y_step64) + (row & 63) * 8;   // Y16[64-row tile][slice][lc][row % 64][8]
        const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(mt * L_pad);
        for (int c0 = 0; c0 < L_pad; c0 += 32) {
          uint32_t v[32];
          tmem_ld32(taddr + c0, v);
          tmem_ld_wait();
          if (row < y_rows_cap) {
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              uint32_t h[4];
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const __half2 p2 = __floats2half2_rn(__uint_as_float(v[8 * g + 2 * i]), __uint_as_float(v[8 * g + 2 * i + 1]));
                h[i] = *reinterpret_cast<const uint32_t*>(&p2);
              }
              *reinterpret_cast<uint4*>(Yt + ((size_t)(c0 >> 3) + g) * 512) = make_uint4(h[0], h[1], h[2], h[3]);
            }
          }
        }
      }
      fence_before();
      mbar_arrive(smem_u32(&acc_empty));
      ++k;
    }
  }
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
F16Plan* f16_plan_create(const SliceParams* sp_host, int n_problems, const SliceParams* fir_host, int n_fir,
                         const BinParams* bp_host, int n_bd, int n_det,
                         int chunk_cap, const double* const* up_w, void* (*q_alloc)(void*, size_t), void* q_ctx,
                         int64_t* bytes, char* err, int errlen)
{
  (void)n_det;
  F16Plan* pl = new F16Plan();
  pl->q_alloc = q_alloc; pl->q_ctx = q_ctx;
  pl->chunk_cap = chunk_cap;
  size_t fixed = 0, stage = 0;
  int gx = 1;
  for (int i = 0; i < n_fir; ++i) {
    const SliceParams& P = fir_host[i];
    if (P.L_pad > 512 || (P.L_pad > 256 && P.L_pad % 32)) { snprintf(err, errlen, "fp16 path: L_pad %d unsupported", P.L_pad); delete pl; return nullptr; }
    int mt = 512 / P.L_pad; mt = mt > 4 ? 4 : (mt < 1 ? 1 : mt);
    const int n_pad = (P.n_taps + FH_KB - 1) / FH_KB * FH_KB;
    const size_t chunks = (size_t)mt * 128 + n_pad;
    const size_t f = chunks * 16 + ((chunks + 16) * 2 + 127) / 128 * 128;
    fixed = f > fixed ? f : fixed;
    const size_t st = (size_t)P.L_pad * FH_KB * 2;
    stage = st > stage ? st : stage;
    const int rows = (chunk_cap >> P.log2d) + P.fir_halo;
    const int g = (rows + 128 * mt - 1) / (128 * mt);
    gx = g > gx ? g : gx;
  }
  const size_t budget = 220 * 1024;
  if (fixed + 2 * stage > budget) { snprintf(err, errlen, "fp16 path: slice too large for shared memory (%zu + 2 x %zu bytes)", fixed, stage); delete pl; return nullptr; }
  int stages = (int)((budget - fixed) / stage);
  if (stages > FH_MAX_STAGES) stages = FH_MAX_STAGES;
  pl->fir_stages = stages;
  pl->fir_smem = (int)(fixed + (size_t)stages * stage);
  pl->fir_grid_x = gx;
  // persistent variant: two Hankel buffers + at least 3 ring stages
  pl->fir_pers = false;
  if (2 * fixed + 3 * stage <= budget) {
    int dev = 0, n_sm = 148;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) n_sm = 148;
    pl->fir_n_sm = n_sm;
    pl->fir_hk_bytes = (int)fixed; pl->fir_stage_cap = (int)stage;
    pl->fir_pers_stages = std::min<int>(FH_MAX_STAGES, (int)((budget - 2 * fixed) / stage));
    pl->fir_pers_smem = (int)(2 * fixed + (size_t)pl->fir_pers_stages * stage);
    size_t cap_units = 0;
    for (int i = 0; i < n_fir; ++i) {
      const SliceParams& P = fir_host[i];
      const int mt = fir_mt_host(P.L_pad);
      const int rows = (chunk_cap >> P.log2d) + P.fir_halo;
      cap_units += (size_t)(rows + 128 * mt - 1) / (128 * mt);
    }
    bool ok = set_max_dyn_smem(fir_f16_pers_kernel) == cudaSuccess;
    pl->fir_cap_units = cap_units;
    for (int k = 0; k < F16Plan::kFirSlots && ok; ++k) {
      void* d = nullptr;
      ok = cudaMalloc(&d, (cap_units + 1) * sizeof(int2)) == cudaSuccess;
      if (ok) { pl->owned.push_back(d); pl->fir_list_dev[k] = d; pl->fir_list_c[k] = -1; *bytes += (int64_t)((cap_units + 1) * sizeof(int2)); }
      if (ok) ok = cudaMallocHost((void**)&pl->fir_list_pin[k], (cap_units + 1) * sizeof(int2)) == cudaSuccess;
      if (ok) ok = cudaEventCreateWithFlags(&pl->fir_list_ev[k], cudaEventDisableTiming) == cudaSuccess;
    }
    pl->fir_pers = ok;
  }
  cudaError_t e = set_max_dyn_smem(fir_f16_kernel);
  if (e != cudaSuccess) { snprintf(err, errlen, "cudaFuncSetAttribute(fir_f16_kernel, %d): %s", pl->fir_smem, cudaGetErrorString(e)); delete pl; return nullptr; }
  if (!f16_plan_build_recon(pl, sp_host, n_problems, bp_host, n_bd, chunk_cap, up_w, bytes, err, errlen)) {
    f16_plan_destroy(pl);
    return nullptr;
  }
  return pl;
}

void f16_plan_destroy(F16Plan* p)
{
  if (!p) return;
  for (int k = 0; k < F16Plan::kFirSlots; ++k) {
    if (p->fir_list_pin[k]) cudaFreeHost(p->fir_list_pin[k]);
    if (p->fir_list_ev[k]) cudaEventDestroy(p->fir_list_ev[k]);
  }
  for (void* q : p->owned) cudaFree(q);
  delete p;
}

// units of one chunk length: sorted by descending cost (taps x tiles), dealt to the CTAs in serpentine order
static int fir_build_list(F16Plan* pl, const SliceParams* sp_host, int n_problems, int c, int slot, cudaStream_t st)
{
  struct Ent { long long cost; int p, r; };
  std::vector<Ent> ents;
  for (int i = 0; i < n_problems; ++i) {
    const SliceParams& P = sp_host[i];
    const int mt = fir_mt_host(P.L_pad);
    const int rows = (c >> P.log2d) + P.fir_halo;
    const int nb = (rows + 128 * mt - 1) / (128 * mt);
    const int n_kb = (P.n_taps + FH_KB - 1) / FH_KB;
    for (int r = 0; r < nb; ++r) {
      const int used = std::min(mt, (rows - r * 128 * mt + 127) / 128);
      ents.push_back(Ent{(long long)n_kb * used * P.L_pad + 40LL * P.L_pad, i, r});
    }
  }
  std::stable_sort(ents.begin(), ents.end(), [](const Ent& a, const Ent& b) { return a.cost > b.cost; });
  if (ents.size() > pl->fir_cap_units) return 1;
  const int G = std::min<int>(pl->fir_n_sm, (int)ents.size());
  if (pl->fir_list_c[slot] >= 0) cudaEventSynchronize(pl->fir_list_ev[slot]);     // the slot's previous upload has left the pinned buffer
  int2* L = pl->fir_list_pin[slot];
  const size_t full = ents.size() / G * G;                  // complete rounds are mirrored on odd rounds, the last partial one is not
  for (size_t i = 0; i < ents.size(); ++i) {
    const size_t round = i / G, j = i % G;
    const size_t pos = (i < full && (round & 1)) ? round * G + (G - 1 - j) : i;
    L[pos] = make_int2(ents[i].p, ents[i].r);
  }
  pl->fir_list_c[slot] = c; pl->fir_list_n[slot] = (int)ents.size();
  if (cudaMemcpyAsync(pl->fir_list_dev[slot], L, ents.size() * sizeof(int2), cudaMemcpyHostToDevice, st) != cudaSuccess) return 1;
  cudaEventRecord(pl->fir_list_ev[slot], st);
  return 0;
}

int launch_fir_f16(F16Plan* pl, const SliceParams* sp_dev, const SliceParams* sp_host, int n_problems,
                   const RateParams* rates_dev, int o, int c, cudaStream_t st, int64_t* launches)
{
  if (pl->fir_pers) {
    // the unit list of this chunk length: cached per length; building one (sort on the host + one async upload from pinned
    // memory) happens the first time a length is seen and is refused while the stream is being captured into a CUDA graph
    int slot = -1;
    for (int k = 0; k < F16Plan::kFirSlots; ++k) if (pl->fir_list_c[k] == c) slot = k;
    if (slot < 0) {
      cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
      cudaStreamIsCapturing(st, &cs);
      if (cs != cudaStreamCaptureStatusNone) { fprintf(stderr, "lloid: graph capture of a chunk length (%d) never filtered before: make one eager call first\n", c); return 1; }
      slot = (c == pl->chunk_cap) ? 0 : 1;
      if (slot) for (int k = 2; k < F16Plan::kFirSlots; ++k) if (pl->fir_list_use[k] < pl->fir_list_use[slot]) slot = k;
      if (fir_build_list(pl, sp_host, n_problems, c, slot, st)) return 1;
    }
    pl->fir_list_use[slot] = ++pl->fir_tick;
    const int n_units = pl->fir_list_n[slot];
    const int grid = std::min(pl->fir_n_sm, n_units);
    fir_f16_pers_kernel<<<grid, FP_THREADS, pl->fir_pers_smem, st>>>(sp_dev, rates_dev, o, c, pl->fir_pers_stages,
                                                                    (const int2*)pl->fir_list_dev[slot], n_units, pl->fir_hk_bytes,
                                                                    pl->fir_stage_cap);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? 0 : 1;
  }
  int gx = 1;
  for (int i = 0; i < n_problems; ++i) {
    const SliceParams& P = sp_host[i];
    int mt = 512 / P.L_pad; mt = mt > 4 ? 4 : (mt < 1 ? 1 : mt);
    const int rows = (c >> P.log2d) + P.fir_halo;
    const int g = (rows + 128 * mt - 1) / (128 * mt);
    gx = g > gx ? g : gx;
  }
  dim3 grid(gx, n_problems);
  fir_f16_kernel<<<grid, FH_THREADS, pl->fir_smem, st>>>(sp_dev, rates_dev, o, c, pl->fir_stages);
  ++*launches;
  return cudaGetLastError() == cudaSuccess ? 0 : 1;
}

}  // namespace lloid
