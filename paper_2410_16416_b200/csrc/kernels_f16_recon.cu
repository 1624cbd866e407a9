// fp16 path (LLOID_F16): A3 reconstruction, A4 upsample + sum and A5 |rho|^2 / windowed maximum on the
// tcgen05 tensor cores (include/lloid.h A3-A5; "matrix multiplication of the orthogonal SNR time
// series with SVD coefficients, and finally up-samples and sums the physical SNR segments").
//
// Two persistent kernels per chunk (one CTA per SM, static cost-balanced (unit, tile) ranges: SchedArgs), built from
// the same pieces: single-thread producer / MMA-issuer roles inside `if (elect_one())`, rings of 8 KB operand stages
// filled by 1-D bulk copies, two TMEM accumulator buffers of 2 x 128 columns so the epilogue of tile t overlaps the
// MMAs of tile t + 1:
//
//  lowrate_recon_kernel   rho^(d)[i, j] = sum_{slices s at rate d} sum_l R^s[i, l] y^s_l[j]     (d > 1)
//      A = R^s (stationary in shared memory for the CTA's 128 templates), B = y^s tiles streamed by two alternating
//      producer threads, D[lane = template, column = low-rate time].  Slices that share a rate are summed BEFORE
//      upsampling (A4 is linear and its kernel depends only on d).  Output Q16: fp16 at the LOW rate, already in
//      the core-matrix layout in which the f0 kernel consumes it as an MMA operand.  The dense f0-rate SNR is
//      never written anywhere.
//
//  f0_kernel   rho[i, k] = sum_{d = 1 slices} R^s y^s  +  sum_{d > 1} rho^(d)[i, window(k)] P_d      then A5
//      The interpolation A4 is itself a tensor-core contraction with the fixed band matrix
//      P_d[r, kl] = d lp_{d,K_up}[...] (16 non-zeros per column), restricted per 16-row chunk to the output
//      columns its band touches.  Cosine and sine rows of a template go to two accumulators (columns
//      [0,128) and [128,256)) of the SAME TMEM lane, so one epilogue thread owns one template: |rho|^2 and
//      the running maximum over time need no cross-lane traffic at all.  Five single-thread roles on two rings
//      (see the comment above f0_kernel).
//
// A single thread retires about one instruction per 7 cycles: per-stage instruction counts of the role loops are
// what bounds the pipeline once the data is there, so the loops carry incrementing ring / pointer / descriptor
// state (no division, no 64-bit descriptor rebuild) and read per-unit tables from shared memory.
#include "f16_plan.h"
#include "tc05.cuh"

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <cstdlib>

namespace lloid {

using namespace tc;

constexpr int RC16_STAGE = 8192;            // bytes per ring stage: one K = 32 (y) or K = 16 (rho^(d)) operand chunk
constexpr int RC16_MAX_STAGES = 16;
constexpr int RC16_SMEM_BUDGET = 219 * 1024;     // + 7 KB static (barriers, tables, epilogue exchange) = 226 of 227 KB

struct LowUnit { int32_t group, rb; };

struct RingBars {
  uint64_t full[RC16_MAX_STAGES], empty[RC16_MAX_STAGES], acc_full[2], acc_empty[2], consts, unit_done;
};

struct Ring {                               // stage index + phase parity, advanced without division
  int s; uint32_t ph; int n;
  __device__ __forceinline__ void advance() { if (++s == n) { s = 0; ph ^= 1u; } }
};

// ---- static persistent schedule (SchedArgs in lloid_internal.h) ------------------------------------
struct SchedPos { int u, t; };              // unit index, first tile

__device__ __forceinline__ SchedPos sched_locate(const SchedArgs& s, long long b)
{
  SchedPos r;
  if (b >= s.cls_base[s.n_cls]) { r.u = s.cls_begin[s.n_cls]; r.t = 0; return r; }
  int c = 0;
  while (c + 1 < s.n_cls && b >= s.cls_base[c + 1]) ++c;
  const long long rem = b - s.cls_base[c];
  const long long nt = s.n_tiles[c];
  int lo = s.cls_begin[c], hi = s.cls_begin[c + 1] - 1;   // largest u with wprefix[u] * nt <= rem
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if ((long long)s.units[mid].wprefix * nt <= rem) lo = mid; else hi = mid - 1;
  }
  const SchedUnit su = s.units[lo];
  r.u = lo; r.t = (int)((rem - (long long)su.wprefix * nt) / su.w);
  return r;
}

// this CTA's range -> rng[0..3] = first unit, first tile, last unit, end tile in the last unit
__device__ __forceinline__ void sched_range(const SchedArgs& s, int* rng)
{
  const long long T = s.cls_base[s.n_cls];
  const SchedPos a = sched_locate(s, T * (long long)blockIdx.x / (long long)gridDim.x);
  const SchedPos b = sched_locate(s, T * (long long)(blockIdx.x + 1) / (long long)gridDim.x);
  rng[0] = a.u; rng[1] = a.t; rng[2] = b.u; rng[3] = b.t;
}

__device__ __forceinline__ int sched_class(const SchedArgs& s, int u)
{
  int c = 0;
  while (c + 1 < s.n_cls && u >= s.cls_begin[c + 1]) ++c;
  return c;
}

__device__ __forceinline__ void ring_setup(RingBars& B, uint32_t* tmem_slot, int n_stages, int warp, int tid, int n_epilogue_threads)
{
  if (warp == 0) tmem_alloc(tmem_slot, 512);
  if (tid == 32) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(smem_u32(&B.full[s]), 1); mbar_init(smem_u32(&B.empty[s]), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(smem_u32(&B.acc_full[b]), 1); mbar_init(smem_u32(&B.acc_empty[b]), n_epilogue_threads); }
    mbar_init(smem_u32(&B.consts), 1);
    mbar_init(smem_u32(&B.unit_done), 1);
    mbar_init_fence();
  }
}

__device__ __forceinline__ void copy_pieces(uint32_t dst, const uint8_t* src, uint32_t bytes, uint32_t bar)
{
  for (uint32_t o = 0; o < bytes; o += 32768u) {
    const uint32_t n = (bytes - o < 32768u) ? bytes - o : 32768u;
    bulk_g2s(dst + o, src + o, n, bar);
  }
}

// The producer and the MMA issuer each run as ONE elected thread inside `if (elect_one())`: ptxas recognises the
// elect.sync-guarded region as single-threaded and keeps the whole loop (ring state, descriptors, barrier
// addresses) in uniform registers -- about 25 SASS instructions per 4-MMA stage, no R2UR at all.  (A per-lane
// predicate on the issuing instruction instead costs an ELECT + R2UR.BROADCAST waterfall per MMA: measured
// ~450 issue cycles per stage, which bounded both kernels.)
// producer: wait for the slot to be free, then one 8 KB bulk copy
__device__ __forceinline__ void produce(Ring& rg, uint32_t bars_full, uint32_t bars_empty, uint32_t ring_base, const uint8_t* src)
{
  mbar_wait(bars_empty + 8u * rg.s, rg.ph ^ 1u);
  mbar_expect_tx(bars_full + 8u * rg.s, RC16_STAGE);
  bulk_g2s(ring_base + (uint32_t)rg.s * RC16_STAGE, src, RC16_STAGE, bars_full + 8u * rg.s);
  rg.advance();
}

// one K = 32 chunk of a reconstruction: D[part] (+)= R[l-groups g .. g + 3][part] * stage^T, N = 128.
// a_lo: descriptor of (group g, part 0) with LBO 4096; b_lo: descriptor of the stage with LBO 2048 (16-byte units)
__device__ __forceinline__ void mma_recon_chunk(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, uint32_t first)
{
  mma_ss(d_tmem,        desc64(a_lo),        desc64(b_lo),        idesc, first ? 0u : 1u);
  mma_ss(d_tmem,        desc64(a_lo + 512u), desc64(b_lo + 256u), idesc, 1u);
  mma_ss(d_tmem + 128u, desc64(a_lo + 128u), desc64(b_lo),        idesc, first ? 0u : 1u);
  mma_ss(d_tmem + 128u, desc64(a_lo + 640u), desc64(b_lo + 256u), idesc, 1u);
}

// ------------------------------------------------------------------------------------------------
struct SegLow {                             // per-role copy of the current unit's operand sources
  const uint8_t* Y[kMaxGroupSlices];
  const uint8_t* Rsrc[kMaxGroupSlices];
  int L[kMaxGroupSlices];
};

__device__ __forceinline__ void seg_low_fill(SegLow& S, const SliceParams* __restrict__ sp, const RateGroup* __restrict__ G, int rb)
{
  for (int i = 0; i < G->n_slices; ++i) {               // one thread
    const SliceParams* P = sp + G->slice[i];
    const int L = P->L_pad;
    S.Y[i] = reinterpret_cast<const uint8_t*>(P->Y);
    S.Rsrc[i] = reinterpret_cast<const uint8_t*>(P->R16) + (size_t)rb * L * 512;
    S.L[i] = L;
  }
}

// Persistent: CTA i of gridDim.x runs cost range i of the (rate, unit, tile) sequence (SchedArgs).  At a unit
// switch the producer first refills the ring with the next unit's y tiles, then waits for the previous unit's
// last accumulator (all MMAs that read the old R are complete) and only then replaces R: the bubble is one R load.
constexpr int LOW_THREADS = 352;             // warps: 0 producer A (+R), 1 MMA issuer, 2-5 epilogue (cos rows), 6 producer B,
                                             // 7-10 epilogue (sin rows): the TMEM -> fp16 -> rho^(d) pass was the slowest stage

__global__ void __launch_bounds__(LOW_THREADS, 1)
lowrate_recon_kernel(const SliceParams* __restrict__ sp, const RateGroup* __restrict__ groups,
                     const LowUnit* __restrict__ units, const __grid_constant__ SchedArgs sched, const __grid_constant__ LowGeom geom)
{
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) RingBars bars;
  __shared__ __align__(8) uint64_t cfull[kNLowRates][RC16_MAX_STAGES], cempty[kNLowRates][RC16_MAX_STAGES], class_go[kNLowRates];
  __shared__ uint32_t tmem_slot;
  __shared__ SegLow seg[3];                             // [0], [2] the producers', [1] MMA issuer's
  __shared__ int s_rng[4];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) sched_range(sched, s_rng);
  __syncthreads();
  const int u_lo = s_rng[0], t_lo = s_rng[1], u_hi = s_rng[2], t_hi = s_rng[3];
  if (u_lo == u_hi && t_lo == t_hi) return;

  ring_setup(bars, &tmem_slot, 0, warp, tid, 256);
  if (tid == 64) {                                      // one ring barrier set per rate class: a CTA visits a class once, and the
    for (int cidx = 0; cidx < kNLowRates; ++cidx) {     // ring geometry (R size, stage count) differs between classes
      for (int st = 0; st < RC16_MAX_STAGES; ++st) { mbar_init(smem_u32(&cfull[cidx][st]), 1); mbar_init(smem_u32(&cempty[cidx][st]), 1); }
      mbar_init(smem_u32(&class_go[cidx]), 1);
    }
    mbar_init_fence();
  }
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem = tmem_slot;
  const uint32_t sR_u = smem_u32(smem);                 // [l_sum / 8][2][128][8] fp16, then the class's ring

  if (warp == 0 || warp == 6) {
    // ===== producers: two elected threads fill alternate stages of the ring (one thread sustains ~1 instruction per
    // 7 cycles: a single producer is slower than the MMAs it feeds); warp 0 also owns R =====
    if (elect_one()) {
    const int pr = warp == 0 ? 0 : 1;
    SegLow& sg = seg[2 * pr];
    Ring rg{0, 0u, 1};
    int own = pr == 0;
    int seg_i = 0, cur_cls = -1;                        // segments done so far by this CTA
    uint32_t bfull = 0, bempty = 0, ring_u = 0;
    for (int u = u_lo; u <= u_hi; ++u) {
      if (u == u_hi && t_hi == 0) break;
      const int cls = sched_class(sched, u);
      const int t0 = (u == u_lo) ? t_lo : 0, t1 = (u == u_hi) ? t_hi : sched.n_tiles[cls];
      if (t0 >= t1) continue;
      const LowUnit un = units[u];
      const RateGroup* G = groups + un.group;
      seg_low_fill(sg, sp, G, un.rb);
      const int ns_u = G->n_slices;
      const uint32_t rbytes_u = (uint32_t)G->l_sum * 512u;
      const bool new_cls = cls != cur_cls;
      if (new_cls) {                                    // other ring geometry: start its ring (and its barrier set) afresh
        cur_cls = cls;
        rg = Ring{0, 0u, geom.n_stages[cls]}; own = pr == 0;
        bfull = smem_u32(&cfull[cls][0]); bempty = smem_u32(&cempty[cls][0]); ring_u = sR_u + (uint32_t)geom.r_bytes[cls];
        // the new ring overlaps the old R / ring: nothing may be written before the previous unit is complete
        if (pr != 0 && seg_i > 0) mbar_wait(smem_u32(&class_go[cls]), 0u);
      }
      const int n_stages = geom.n_stages[cls];
      int countdown = (seg_i == 0 || new_cls) ? 0 : n_stages;      // ring stages to push before R is replaced
      bool r_done = pr != 0;
      auto load_R = [&]() {
        // every MMA that reads the old R is complete.  (A parity wait on acc_full is not usable here: with short tiles the
        // producer runs several accumulator phases ahead and the parity would alias; this barrier is at most one phase away.)
        if (seg_i > 0) mbar_wait(smem_u32(&bars.unit_done), (uint32_t)(seg_i - 1) & 1u);
        if (new_cls && seg_i > 0) mbar_arrive(smem_u32(&class_go[cls]));      // producer B may start on the new ring
        {
          mbar_expect_tx(smem_u32(&bars.consts), rbytes_u);
          uint32_t off = 0;
          for (int i = 0; i < ns_u; ++i) {
            copy_pieces(sR_u + off, sg.Rsrc[i], (uint32_t)sg.L[i] * 512u, smem_u32(&bars.consts));
            off += (uint32_t)sg.L[i] * 512u;
          }
        }
        r_done = true;
      };
      if (!r_done && countdown == 0) load_R();
      for (int t = t0; t < t1; ++t)
        for (int i = 0; i < ns_u; ++i) {
          const int L = sg.L[i];
          const uint8_t* src = sg.Y[i] + (size_t)t * L * 256;          // tiles are contiguous in Y16
          for (int kc = 0; kc < (L >> 5); ++kc, src += RC16_STAGE) {
            if (own) produce(rg, bfull, bempty, ring_u, src); else rg.advance();
            own ^= 1;
            if (!r_done && --countdown == 0) load_R();
          }
        }
      if (!r_done) load_R();
      ++seg_i;
    }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: one elected thread =====
    if (elect_one()) {
    const uint32_t idesc = idesc_f16(128, 128);
    const uint32_t a_base = desc_lo(sR_u, 4096u);
    const uint32_t tm = tmem;
    Ring rg{0, 0u, 1};
    int cur_cls = -1;
    uint32_t bfull = 0, bempty = 0, b_base = 0;
    uint32_t eph = 3u;                                  // bit buf: parity to wait for on acc_empty (first use: free)
    int buf = 0, seg_i = 0;
    for (int u = u_lo; u <= u_hi; ++u) {
      if (u == u_hi && t_hi == 0) break;
      const int cls = sched_class(sched, u);
      const int t0 = (u == u_lo) ? t_lo : 0, t1 = (u == u_hi) ? t_hi : sched.n_tiles[cls];
      if (t0 >= t1) continue;
      const LowUnit un = units[u];
      const RateGroup* G = groups + un.group;
      seg_low_fill(seg[1], sp, G, un.rb);
      const int ns_u = G->n_slices;
      if (cls != cur_cls) {
        cur_cls = cls;
        rg = Ring{0, 0u, geom.n_stages[cls]};
        bfull = smem_u32(&cfull[cls][0]); bempty = smem_u32(&cempty[cls][0]);
        b_base = desc_lo(sR_u + (uint32_t)geom.r_bytes[cls], 2048u);
      }
      mbar_wait(smem_u32(&bars.consts), (uint32_t)seg_i & 1u);
      fence_after();
      for (int t = t0; t < t1; ++t, buf ^= 1) {
        mbar_wait(smem_u32(&bars.acc_empty[buf]), (eph >> buf) & 1u); eph ^= 1u << buf;
        fence_after();
        const uint32_t d_tmem = tm + (uint32_t)(buf * 256);
        uint32_t first = 1u, a_lo = a_base;
        for (int i = 0; i < ns_u; ++i) {
          const int n_kc = seg[1].L[i] >> 5;
          for (int kc = 0; kc < n_kc; ++kc, a_lo += 1024u) {
            mbar_wait(bfull + 8u * rg.s, rg.ph);
            fence_after();
            mma_recon_chunk(d_tmem, a_lo, b_base + (uint32_t)rg.s * (RC16_STAGE / 16), idesc, first);
            commit(bempty + 8u * rg.s);
            first = 0u;
            rg.advance();
          }
        }
        commit(smem_u32(&bars.acc_full[buf]));
      }
      commit(smem_u32(&bars.unit_done));
      ++seg_i;
    }
    }
  } else {
    // ===== epilogue: warps 2-5 convert the cosine accumulator, warps 7-10 the sine one (lane quarter = warp % 4) =====
    const int q = warp & 3;
    const int pl = q * 32 + lane;
    const int part = warp >= 7 ? 1 : 0;
    uint32_t fph = 0u;
    int buf = 0;
    for (int u = u_lo; u <= u_hi; ++u) {
      if (u == u_hi && t_hi == 0) break;
      const int cls = sched_class(sched, u);
      const int t0 = (u == u_lo) ? t_lo : 0, t1 = (u == u_hi) ? t_hi : sched.n_tiles[cls];
      if (t0 >= t1) continue;
      const LowUnit un = units[u];
      const RateGroup* Gp = groups + un.group;
      __half* __restrict__ Q = Gp->Q;
      const int q_cap = Gp->q_groups_cap;
      for (int t = t0; t < t1; ++t, buf ^= 1) {
        mbar_wait(smem_u32(&bars.acc_full[buf]), (fph >> buf) & 1u); fph ^= 1u << buf;
        fence_after();
        const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 256);
#pragma unroll 1
          for (int c0 = 0; c0 < 128; c0 += 32) {
            uint32_t v[32];
            tmem_ld32(taddr + (uint32_t)(part * 128 + c0), v);
            tmem_ld_wait();
#pragma unroll
            for (int gq = 0; gq < 4; ++gq) {
              uint32_t h[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                const __half2 p2 = __floats2half2_rn(__uint_as_float(v[8 * gq + 2 * e]), __uint_as_float(v[8 * gq + 2 * e + 1]));
                h[e] = *reinterpret_cast<const uint32_t*>(&p2);
              }
              const int jg = t * 16 + (c0 >> 3) + gq;
              if (jg < q_cap)
                *reinterpret_cast<uint4*>(Q + ((((size_t)un.rb * q_cap + jg) * 2 + part) * 128 + pl) * 8) =
                    make_uint4(h[0], h[1], h[2], h[3]);
            }
          }
        fence_before();
        mbar_arrive(smem_u32(&bars.acc_empty[buf]));
      }
    }
  }
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
struct F0Args {
  const SliceParams* sp; const BdPlan* bd; const F0Combo* combos; const RateGroup* groups; const uint8_t* P;
  Peak* partials; Capture cap; long long k_a;
  int n_lr, c, r_bytes, r_bufs, tiles_cap, max_templates, nsy, nsq, p_bytes;
  SchedArgs sched;                                      // units = combos, one class
  UpRate up[kNLowRates];
  QItem item[kNLowRates][2][8];                         // per rate and variant: the active 16-row chunks, in order (kernel
  int32_t n_items[kNLowRates][2];                       // parameters: read with uniform loads); QItem.ch = chunk index
};

struct SegF0 {                                          // per-role copy of the current unit's operand sources
  const uint8_t* Y[kMaxF0Slices];
  const uint8_t* Rsrc[kMaxF0Slices];
  int L[kMaxF0Slices];
  const uint8_t* Q[kNLowRates];                         // this template block's rho^(d), or null
};

__device__ __forceinline__ void seg_f0_fill(SegF0& S, const F0Args& a, const F0Combo cb, const BdPlan* __restrict__ B)
{
  for (int i = 0; i < B->n_f0; ++i) {                   // one thread
    const SliceParams* P = a.sp + B->f0_slice[i];
    const int L = P->L_pad;
    S.Y[i] = reinterpret_cast<const uint8_t*>(P->Y);
    S.Rsrc[i] = reinterpret_cast<const uint8_t*>(P->R16) + (size_t)cb.rb * L * 512;
    S.L[i] = L;
  }
  for (int r = 0; r < a.n_lr; ++r) {
    const RateGroup* G = a.groups + cb.bd * a.n_lr + r;
    S.Q[r] = (G->n_slices > 0) ? reinterpret_cast<const uint8_t*>(G->Q) + (size_t)cb.rb * G->q_groups_cap * 4096 : nullptr;
  }
}

// Per-unit tables of the interpolation work of one tile, so that the per-chunk code of the single-thread loops
// is a table read plus the issuing instructions.  v = t & 1 selects the band-matrix variant of the rates whose
// window start alternates (d = 32); the chunks of a (rate, variant) are consecutive.
struct ItTab { uint32_t idesc, b_lo, d_off, pad; };                                  // MMA issuer: one per chunk
struct PrTab { const uint8_t* q; int32_t log2d, ch0[2], n[2]; int32_t pad; };           // producer: one per rate present
constexpr int kMaxTileItems = kNLowRates * 8;

// f0_kernel roles.  A single thread sustains one instruction every ~7 cycles, so one producer and one issuer
// thread cannot feed 19 eight-KB stages per 2600-cycle tile; the work is split over five single-thread roles
// over two rings (y tiles: PY -> IY; window chunks: PQ0 / PQ1 alternate -> IQ).  Each ring has ONE consumer, so its
// slots are released in order and a producer can never run two laps ahead of a slot (which would alias the
// barrier's phase parity):
//   warp 0  PY   bulk copies of the y tiles of the d = 1 slices; owns R and P (stationary operands)
//   warp 6,7 PQ  bulk copies of the rho^(d) window chunks, even / odd chunk of the tile
//   warp 1  IY   MMAs of the d = 1 slices into accumulator buf = tile parity, then commit -> ybar[buf]
//   warp 8  IQ   waits ybar[buf] (the y part is COMPLETE: orders its accumulating MMAs after IY's zeroing one),
//                interpolation MMAs, commit -> acc_full[buf]
//   warps 2-5    epilogue, columns [0, 64) of the tile (one thread = one template)
//   warps 9-12   epilogue, columns [64, 128); hands its partial maximum to the first group through shared memory.
//                With L = 64 (config 3) the MMAs of a tile take ~1000 cycles and a single 128-column epilogue pass
//                ~2900: the kernel ran at the epilogue's pace.
// While IQ works on tile t, IY already fills the other accumulator with tile t + 1.
constexpr int F0_THREADS = 416;

struct F0Bars {
  uint64_t full[RC16_MAX_STAGES], empty[RC16_MAX_STAGES];      // y ring: slots [0, nsy); chunk ring: slots [nsy, nsy + nsq)
  uint64_t acc_full[2], acc_empty[2], ybar[2], consts[2], unit_done[2];
};

#define FOR_SEGMENTS(u, t0, t1)                                                                   \
  for (int u = u_lo; u <= u_hi; ++u)                                                              \
    if (u == u_hi && t_hi == 0) break;                                                            \
    else if (const int t0 = (u == u_lo) ? t_lo : 0, t1 = (u == u_hi) ? t_hi : n_tiles; t0 >= t1) continue; \
    else

// stages of one tile of this unit: y chunks, interpolation chunks per variant
__device__ __forceinline__ void f0_unit_counts(const F0Args& a, const F0Combo cb, const BdPlan* __restrict__ B, int& ny, int (&nit)[2])
{
  ny = B->l_sum >> 5;
  nit[0] = nit[1] = 0;
  for (int r = 0; r < a.n_lr; ++r) {
    if (a.groups[cb.bd * a.n_lr + r].n_slices == 0) continue;
    nit[0] += a.n_items[r][0];
    nit[1] += a.n_items[r][a.up[r].n_var > 1 ? 1 : 0];
  }
}

__global__ void __launch_bounds__(F0_THREADS, 1)
f0_kernel(const __grid_constant__ F0Args a)
{
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) F0Bars bars;
  __shared__ uint32_t tmem_slot;
  __shared__ SegF0 seg[2];                              // [0] PY's, [1] IY's
  __shared__ __align__(16) ItTab s_it[2][kMaxTileItems];
  __shared__ PrTab s_pr[2][kNLowRates];
  __shared__ int s_rng[4];
  __shared__ __align__(16) uint4 s_qst[RC16_MAX_STAGES];   // IQ: per chunk-ring stage {operand descriptor, full barrier, empty barrier}
  __shared__ __align__(16) Peak s_half[2][kTplBlock];    // second column half's partial maximum, per accumulator buffer

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) sched_range(a.sched, s_rng);
  __syncthreads();
  const int u_lo = s_rng[0], t_lo = s_rng[1], u_hi = s_rng[2], t_hi = s_rng[3];
  if (u_lo == u_hi && t_lo == t_hi) return;
  const int n_tiles = a.sched.n_tiles[0];

  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  if (tid == 32) {
    for (int s = 0; s < RC16_MAX_STAGES; ++s) { mbar_init(smem_u32(&bars.full[s]), 1); mbar_init(smem_u32(&bars.empty[s]), 1); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(smem_u32(&bars.acc_full[b]), 1); mbar_init(smem_u32(&bars.acc_empty[b]), 256);
      mbar_init(smem_u32(&bars.ybar[b]), 1); mbar_init(smem_u32(&bars.consts[b]), 1); mbar_init(smem_u32(&bars.unit_done[b]), 1);
    }
    mbar_init_fence();
  }
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem = tmem_slot;
  const int n_lr = a.n_lr;
  const int nsy = a.nsy, nsq = a.nsq;
  const int r_bufs = a.r_bufs;
  const uint32_t bfull = smem_u32(&bars.full[0]), bempty = smem_u32(&bars.empty[0]);
  const uint32_t qfull = bfull + 8u * nsy, qempty = bempty + 8u * nsy;
  const uint32_t sR_u = smem_u32(smem);                 // r_bufs x [l_sum / 8][2][128][8] fp16
  const uint32_t sP_u = sR_u + (uint32_t)(a.r_bytes * r_bufs);   // band matrices
  const uint32_t ring_u = sP_u + (uint32_t)a.p_bytes;
  const uint32_t qring_u = ring_u + (uint32_t)nsy * RC16_STAGE;

  if (warp == 0) {
    // ===== PY: y tiles of the d = 1 slices, R and P =====
    if (elect_one()) {
      int seg_i = 0;
      Ring rg{0, 0u, nsy};
      FOR_SEGMENTS(u, t0, t1) {
        const F0Combo cb = a.combos[u];
        const BdPlan* B = a.bd + cb.bd;
        seg_f0_fill(seg[0], a, cb, B);
        const int nf_u = B->n_f0;
        const int rb_i = seg_i % r_bufs, use = seg_i / r_bufs;
        // R (and P, once) go out after `pre` y stages of the unit's first tile are in flight: the ring refills while
        // the previous unit drains, and the switch costs one R load.  pre <= ring size, or IY (which waits for R) could
        // never free the slot PY is waiting for.
        int pre = (seg_i == 0) ? 0 : min(nsy, B->l_sum >> 5);
        bool need_R = true;
        auto load_R = [&]() {
          // this R buffer's previous unit is complete (per-buffer barrier: never more than one phase away)
          if (use > 0) mbar_wait(smem_u32(&bars.unit_done[rb_i]), (uint32_t)(use - 1) & 1u);
          const uint32_t cb_u = smem_u32(&bars.consts[rb_i]);
          mbar_expect_tx(cb_u, (uint32_t)B->l_sum * 512u + (seg_i == 0 ? (uint32_t)a.p_bytes : 0u));
          uint32_t off = (uint32_t)(rb_i * a.r_bytes);
          for (int i = 0; i < nf_u; ++i) {
            copy_pieces(sR_u + off, seg[0].Rsrc[i], (uint32_t)seg[0].L[i] * 512u, cb_u);
            off += (uint32_t)seg[0].L[i] * 512u;
          }
          if (seg_i == 0) copy_pieces(sP_u, a.P, (uint32_t)a.p_bytes, cb_u);
          need_R = false;
        };
        if (pre == 0) load_R();
        for (int t = t0; t < t1; ++t)
          for (int i = 0; i < nf_u; ++i) {
            const int L = seg[0].L[i];
            const uint8_t* src = seg[0].Y[i] + (size_t)t * L * 256;      // tiles are contiguous in Y16
            for (int kc = 0; kc < (L >> 5); ++kc, src += RC16_STAGE) {
              produce(rg, bfull, bempty, ring_u, src);
              if (need_R && --pre == 0) load_R();
            }
          }
        ++seg_i;
      }
    }
  } else if (warp == 6 || warp == 7) {
    // ===== PQ: rho^(d) window chunks, even (warp 6) / odd (warp 7) chunk of the tile =====
    if (elect_one()) {
      const int pq = warp - 6;
      PrTab* tab = s_pr[pq];
      Ring rg{0, 0u, nsq};
      int own = pq == 0;                                 // the ring's stages alternate between the two PQ threads
      FOR_SEGMENTS(u, t0, t1) {
        const F0Combo cb = a.combos[u];
        int npr = 0;
        for (int r = 0; r < n_lr; ++r) {
          const RateGroup* G = a.groups + cb.bd * n_lr + r;
          if (G->n_slices == 0) continue;
          PrTab e;
          e.q = reinterpret_cast<const uint8_t*>(G->Q) + (size_t)cb.rb * G->q_groups_cap * 4096;
          e.log2d = a.up[r].log2d; e.pad = 0;
          for (int v = 0; v < 2; ++v) {
            const int vv = a.up[r].n_var > 1 ? v : 0;
            e.n[v] = a.n_items[r][vv];
            e.ch0[v] = e.n[v] > 0 ? (int)a.item[r][vv][0].ch : 0;
          }
          tab[npr++] = e;
        }
        for (int t = t0; t < t1; ++t) {
          const int v = t & 1;
          for (int j = 0; j < npr; ++j) {
            const PrTab* e = &tab[j];
            const int ws = ((t * 128) >> e->log2d) & ~7;
            const uint8_t* src = e->q + (size_t)(ws >> 3) * 4096 + (size_t)e->ch0[v] * RC16_STAGE;
            const int n_it = e->n[v];
            for (int i = 0; i < n_it; ++i, src += RC16_STAGE, own ^= 1) {
              if (own) produce(rg, qfull, qempty, qring_u, src); else rg.advance();
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===== IY: MMAs of the d = 1 slices =====
    if (elect_one()) {
      const uint32_t idesc128 = idesc_f16(128, 128);
      const uint32_t a_base = desc_lo(sR_u, 4096u), b_base = desc_lo(ring_u, 2048u);
      uint32_t eph = 3u;                                  // bit buf: parity to wait for on acc_empty (first use: free)
      int seg_i = 0, buf = 0;
      Ring rg{0, 0u, nsy};
      FOR_SEGMENTS(u, t0, t1) {
        const F0Combo cb = a.combos[u];
        const BdPlan* B = a.bd + cb.bd;
        seg_f0_fill(seg[1], a, cb, B);
        const int nf_u = B->n_f0;
        const int rb_i = seg_i % r_bufs, use = seg_i / r_bufs;
        mbar_wait(smem_u32(&bars.consts[rb_i]), (uint32_t)use & 1u);
        fence_after();
        const uint32_t a_seg = a_base + (uint32_t)((rb_i * a.r_bytes) >> 4);
        for (int t = t0; t < t1; ++t, buf ^= 1) {
          mbar_wait(smem_u32(&bars.acc_empty[buf]), (eph >> buf) & 1u); eph ^= 1u << buf;
          fence_after();
          const uint32_t d_tmem = tmem + (uint32_t)(buf * 256);
          uint32_t first = 1u, a_lo = a_seg;
          for (int i = 0; i < nf_u; ++i) {
            const int n_kc = seg[1].L[i] >> 5;
            for (int kc = 0; kc < n_kc; ++kc, a_lo += 1024u) {
              mbar_wait(bfull + 8u * rg.s, rg.ph);
              fence_after();
              mma_recon_chunk(d_tmem, a_lo, b_base + (uint32_t)rg.s * (RC16_STAGE / 16), idesc128, first);
              commit(bempty + 8u * rg.s);
              first = 0u;
              rg.advance();
            }
          }
          commit(smem_u32(&bars.ybar[buf]));
        }
        ++seg_i;
      }
    }
  } else if (warp == 8) {
    // ===== IQ: interpolation MMAs (A4), after the tile's y part is complete =====
    if (elect_one()) {
      const uint32_t qa_base = desc_lo(qring_u, 4096u), p_base = desc_lo(sP_u, 2048u);
      uint32_t yph = 0u;
      int seg_i = 0, buf = 0;
      Ring rg{0, 0u, nsq};
      // Everything a chunk needs is read from two small tables (one LDS.128 each) instead of being recomputed: every
      // value the MMA takes has to cross from a vector to a uniform register (R2UR), and this loop is the kernel's
      // critical path.
      for (int st = 0; st < nsq; ++st)
        s_qst[st] = make_uint4(qa_base + (uint32_t)st * (RC16_STAGE / 16), qfull + 8u * st, qempty + 8u * st, 0u);
      FOR_SEGMENTS(u, t0, t1) {
        const F0Combo cb = a.combos[u];
        const BdPlan* B = a.bd + cb.bd;
        int nit[2] = {0, 0};
        for (int v = 0; v < 2; ++v)
          for (int r = 0; r < n_lr; ++r) {
            if (a.groups[cb.bd * n_lr + r].n_slices == 0) continue;
            const int vv = a.up[r].n_var > 1 ? v : 0;
            for (int i = 0; i < a.n_items[r][vv]; ++i) {
              const QItem it = a.item[r][vv][i];
              // tiles of parity v use accumulator buf ^ ((v ^ t0) & 1): the accumulator address goes into the table
              ItTab e; e.idesc = it.idesc; e.b_lo = p_base + it.b_off; e.pad = 0;
              e.d_off = tmem + (uint32_t)((buf ^ ((v ^ t0) & 1)) * 256) + it.d_off;
              s_it[v][nit[v]++] = e;
            }
          }
        const int rb_i = seg_i % r_bufs, use = seg_i / r_bufs;
        if (seg_i == 0) { mbar_wait(smem_u32(&bars.consts[0]), 0u); fence_after(); }   // P has landed (loaded once, with the first R)
        for (int t = t0; t < t1; ++t, buf ^= 1) {
          mbar_wait(smem_u32(&bars.ybar[buf]), (yph >> buf) & 1u); yph ^= 1u << buf;
          fence_after();
          const ItTab* tab = s_it[t & 1];
          const int n_it = nit[t & 1];
          for (int k = 0; k < n_it; ++k) {
            const uint4 e = *reinterpret_cast<const uint4*>(tab + k);     // idesc, b_lo, accumulator address
            const uint4 q = s_qst[rg.s];                                  // operand descriptor, full, empty barrier
            mbar_wait(q.y, rg.ph);
            fence_after();
            const uint64_t bdesc = desc64(e.y);
            mma_ss(e.z,        desc64(q.x),        bdesc, e.x, 1u);
            mma_ss(e.z + 128u, desc64(q.x + 128u), bdesc, e.x, 1u);
            commit(q.z);
            rg.advance();
          }
          commit(smem_u32(&bars.acc_full[buf]));
        }
        commit(smem_u32(&bars.unit_done[rb_i]));
        (void)use;
        ++seg_i;
      }
    }
  } else if ((warp >= 2 && warp <= 5) || warp >= 9) {
    // ===== epilogue: one thread = one template and one half of the tile's columns; |rho|^2 and first maximum =====
    const int q = warp & 3;                           // TMEM lane quarter this warp may access
    const int half = warp >= 9 ? 1 : 0;
    const int pl = q * 32 + lane;
    uint32_t fph = 0u;
    int buf = 0;
    FOR_SEGMENTS(u, t0, t1) {
      const F0Combo cb = a.combos[u];
      const int n_templates = a.bd[cb.bd].n_templates;
      const int p = cb.rb * kTplBlock + pl;
      const bool capture = a.cap.snr != nullptr && a.cap.bd == cb.bd && 2 * p + 1 < a.cap.rows;
      for (int t = t0; t < t1; ++t, buf ^= 1) {
        mbar_wait(smem_u32(&bars.acc_full[buf]), (fph >> buf) & 1u); fph ^= 1u << buf;
        fence_after();
        const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 256);
        const int kap0 = t * 128;
        const int valid = min(128, a.c - kap0);
        // four interleaved running maxima (columns j = m mod 4) break the serial compare/select chain; merged below
        // with "larger q, then lower k" so that the first maximum of the tile still wins (R8)
        float bq[4] = {-1.f, -1.f, -1.f, -1.f}, bre4[4] = {0.f, 0.f, 0.f, 0.f}, bim4[4] = {0.f, 0.f, 0.f, 0.f};
        int bk4[4] = {0, 0, 0, 0};
  #pragma unroll 1
        for (int c0 = 64 * half; c0 < 64 * half + 64; c0 += 32) {
          uint32_t re[32], im[32];
          tmem_ld32(taddr + (uint32_t)c0, re);
          tmem_ld32(taddr + (uint32_t)(128 + c0), im);
          tmem_ld_wait();
          if (c0 + 32 <= valid) {
  #pragma unroll
            for (int j = 0; j < 32; ++j) {
              const float x = __uint_as_float(re[j]), y = __uint_as_float(im[j]);
              const float qq = fmaf(x, x, y * y);
              if (qq > bq[j & 3]) { bq[j & 3] = qq; bk4[j & 3] = c0 + j; bre4[j & 3] = x; bim4[j & 3] = y; }
            }
          } else {
  #pragma unroll
            for (int j = 0; j < 32; ++j) {
              const float x = __uint_as_float(re[j]), y = __uint_as_float(im[j]);
              const float qq = fmaf(x, x, y * y);
              if (c0 + j < valid && qq > bq[j & 3]) { bq[j & 3] = qq; bk4[j & 3] = c0 + j; bre4[j & 3] = x; bim4[j & 3] = y; }
            }
          }
          if (capture) {
  #pragma unroll
            for (int j = 0; j < 32; ++j) {
              const long long k = a.k_a + kap0 + c0 + j;
              if (c0 + j < valid && k >= a.cap.k_begin && k < a.cap.k_begin + a.cap.n) {
                a.cap.snr[(size_t)(2 * p) * a.cap.n + (k - a.cap.k_begin)] = __uint_as_float(re[j]);
                a.cap.snr[(size_t)(2 * p + 1) * a.cap.n + (k - a.cap.k_begin)] = __uint_as_float(im[j]);
              }
            }
          }
        }
        float best = bq[0], bre = bre4[0], bim = bim4[0];
        int bk = bk4[0];
  #pragma unroll
        for (int m = 1; m < 4; ++m)
          if (bq[m] > best || (bq[m] == best && bk4[m] < bk)) { best = bq[m]; bk = bk4[m]; bre = bre4[m]; bim = bim4[m]; }
        fence_before();
        mbar_arrive(smem_u32(&bars.acc_empty[buf]));
        // s_half[buf] of tile t is rewritten at tile t + 2, i.e. after the barrier of tile t + 1, which the first group
        // reaches only after it has read tile t's entry
        if (half) { Peak pk; pk.q = best; pk.kappa = bk; pk.re = bre; pk.im = bim; s_half[buf][pl] = pk; }
        asm volatile("bar.sync 2, 256;" ::: "memory");
        if (!half) {
          const Peak o = s_half[buf][pl];
          if (o.q > best) { best = o.q; bk = o.kappa; bre = o.re; bim = o.im; }   // its columns are later: ties stay with the first half
          if (p < n_templates) {
            Peak pk; pk.q = best; pk.kappa = kap0 + bk; pk.re = bre; pk.im = bim;
            a.partials[((size_t)cb.bd * a.tiles_cap + t) * a.max_templates + p] = pk;
          }
        }
      }
    }
  }
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}
// ------------------------------------------------------------------------------------------------
// host side: plan
// ------------------------------------------------------------------------------------------------
namespace {

bool plan_alloc(F16Plan* pl, void** p, size_t n, bool zero, int64_t* bytes, char* err, int errlen)
{
  if (n == 0) n = 16;
  cudaError_t e = cudaMalloc(p, n);
  if (e == cudaSuccess && zero) e = cudaMemset(*p, 0, n);
  if (e != cudaSuccess) { snprintf(err, errlen, "fp16 plan: device allocation of %zu bytes failed: %s", n, cudaGetErrorString(e)); return false; }
  pl->owned.push_back(*p);
  *bytes += (int64_t)n;
  return true;
}

}  // namespace

bool f16_plan_build_recon(F16Plan* pl, const SliceParams* sp_host, int n_problems, const BinParams* bp_host,
                          int n_bd, int chunk_cap, const double* const* up_w, int64_t* bytes, char* err, int errlen)
{
  (void)n_problems;
  pl->tensor_recon = false;
  pl->n_bd = n_bd;
  int dev = 0, n_sm = 148;
  cudaGetDevice(&dev);
  if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n_sm > 0) pl->n_sm = n_sm;

  // distinct low rates, ascending d
  bool have[kMaxRates] = {false, false, false, false, false, false};
  for (int b = 0; b < n_bd; ++b)
    for (int s = 0; s < bp_host[b].n_slices; ++s) have[sp_host[bp_host[b].first_slice + s].log2d] = true;
  int lr_of[kMaxRates];
  pl->n_lr = 0;
  for (int l2 = 1; l2 < kMaxRates; ++l2) { lr_of[l2] = -1; if (have[l2]) { lr_of[l2] = pl->n_lr; pl->up[pl->n_lr].log2d = l2; ++pl->n_lr; } }

  // A (bin, detector) the tensor kernels cannot hold is EXCLUDED from their work lists and reconstructed by the FFMA
  // kernels (lloid_api.cu); the others stay on the tensor path.
  pl->excluded.assign(n_bd, 0);
  pl->bd_host.assign(n_bd, BdPlan());
  pl->groups_host.assign((size_t)n_bd * std::max(pl->n_lr, 1), RateGroup());
  pl->combos_host.clear();
  pl->l_sum_f0_max = pl->l_sum_low_max = 0;
  for (int b = 0; b < n_bd; ++b) {
    bool ok = true;
    BdPlan& B = pl->bd_host[b];
    memset(&B, 0, sizeof B);
    B.n_templates = bp_host[b].n_templates;
    B.n_rb = (B.n_templates + kTplBlock - 1) / kTplBlock;
    for (int r = 0; r < pl->n_lr; ++r) {
      RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + r];
      memset(&G, 0, sizeof G);
      G.log2d = pl->up[r].log2d; G.n_rb = B.n_rb;
      G.q_groups_cap = (((chunk_cap >> G.log2d) + 2 * kKUp + 127) / 128) * 16 + 16;
    }
    for (int s = 0; s < bp_host[b].n_slices; ++s) {
      const int idx = bp_host[b].first_slice + s;
      const SliceParams& P = sp_host[idx];
      if (P.rows_pad != B.n_rb * 2 * kTplBlock || P.L_pad % 32) { ok = false; break; }
      if (P.d == 1) {
        if (B.n_f0 == kMaxF0Slices) { ok = false; break; }
        B.f0_slice[B.n_f0++] = idx; B.l_sum += P.L_pad;
      } else {
        RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + lr_of[P.log2d]];
        if (G.n_slices == kMaxGroupSlices) { ok = false; break; }
        G.slice[G.n_slices++] = idx; G.l_sum += P.L_pad;
      }
    }
    if (B.n_f0 == 0) ok = false;
    if (!ok) pl->excluded[b] = 1;
  }

  // band matrices P_d (A4):  c[kl] = sum_r Q[ws + r] P[r, kl],  ws = (128 t / d) & ~7, mis = 128 t / d - ws,
  // P[r, kl] = w_phi[i], i = mis + floor(kl / d) + K_up - r in [-K_up, K_up), phi = kl mod d
  std::vector<__half> pblob;
  for (int r = 0; r < pl->n_lr; ++r) {
    UpRate& U = pl->up[r];
    const int d = 1 << U.log2d;
    if (!up_w || !up_w[U.log2d]) return true;
    const double* w = up_w[U.log2d];
    U.n_var = (128 / d) % 8 ? 2 : 1;
    const int mis_max = (U.n_var == 2) ? 128 / d : 0;
    U.k_win = (128 / d + 2 * kKUp + mis_max + 15) / 16 * 16;
    if (U.k_win / 16 > 8) return true;
    memset(U.n0, 0, sizeof U.n0); memset(U.nn, 0, sizeof U.nn);
    U.p_off[1] = 0;
    for (int v = 0; v < U.n_var; ++v) {
      const int mis = v * mis_max;
      U.p_off[v] = (int)(pblob.size() * sizeof(__half));
      const size_t base = pblob.size();
      pblob.resize(base + (size_t)U.k_win * 128, __float2half(0.f));
      std::vector<int> cmin(U.k_win / 16, 1 << 30), cmax(U.k_win / 16, -1);
      for (int rw = 0; rw < U.k_win; ++rw)
        for (int kl = 0; kl < 128; ++kl) {
          const int i = mis + kl / d + kKUp - rw;
          if (i < -kKUp || i >= kKUp) continue;
          pblob[base + ((size_t)(rw >> 3) * 128 + kl) * 8 + (rw & 7)] = __float2half_rn((float)w[(size_t)(i + kKUp) * d + kl % d]);
          cmin[rw >> 4] = std::min(cmin[rw >> 4], kl); cmax[rw >> 4] = std::max(cmax[rw >> 4], kl);
        }
      for (int ch = 0; ch < U.k_win / 16; ++ch) {
        if (cmax[ch] < 0) continue;
        int n0 = cmin[ch] / 8 * 8;
        const int nn = (cmax[ch] + 1 - n0 + 15) / 16 * 16;
        if (n0 + nn > 128) n0 = 128 - nn;
        U.n0[v][ch] = (uint8_t)(n0 / 8); U.nn[v][ch] = (uint8_t)(nn / 8);
      }
    }
  }
  pl->p_bytes = (int)(pblob.size() * sizeof(__half));
  for (int r = 0; r < pl->n_lr; ++r)                       // the kernels rely on: active chunks of a variant are consecutive,
    for (int v = 0; v < pl->up[r].n_var; ++v) {            // and only a window start that alternates with t has two variants
      int first = -1, last = -1, cnt = 0;
      for (int ch = 0; ch < (pl->up[r].k_win >> 4); ++ch)
        if (pl->up[r].nn[v][ch]) { if (first < 0) first = ch; last = ch; ++cnt; }
      if (cnt == 0 || last - first + 1 != cnt) return true;
    }

  // per-bin shared-memory limits: stationary R (single-buffered) + P + 4 ring stages / stationary R + 4 ring stages
  {
    const int lim_f0 = (RC16_SMEM_BUDGET - pl->p_bytes - 4 * RC16_STAGE) / 512;
    const int lim_low = (RC16_SMEM_BUDGET - 4 * RC16_STAGE) / 512;
    for (int b = 0; b < n_bd; ++b) {
      if (pl->bd_host[b].l_sum > lim_f0) pl->excluded[b] = 1;
      for (int r = 0; r < pl->n_lr; ++r)
        if (pl->groups_host[(size_t)b * pl->n_lr + r].l_sum > lim_low) pl->excluded[b] = 1;
      if (pl->excluded[b]) { pl->any_excluded = true; continue; }
      pl->l_sum_f0_max = std::max(pl->l_sum_f0_max, pl->bd_host[b].l_sum);
      for (int r = 0; r < pl->n_lr; ++r) pl->l_sum_low_max = std::max(pl->l_sum_low_max, pl->groups_host[(size_t)b * pl->n_lr + r].l_sum);
      for (int rb = 0; rb < pl->bd_host[b].n_rb; ++rb) pl->combos_host.push_back(F0Combo{b, rb});
    }
    if (pl->combos_host.empty()) return true;             // nothing fits: the whole bank goes to the FFMA kernels
  }

  // shared-memory budgets (operands stationary: R of the CTA's template block, and P)
  // R double-buffered (no bubble at a unit switch) when that still leaves >= 8 ring stages
  pl->f0_r_bufs = (RC16_SMEM_BUDGET - 2 * pl->l_sum_f0_max * 512 - pl->p_bytes) / RC16_STAGE >= 8 ? 2 : 1;
  const int f0_fixed = pl->f0_r_bufs * pl->l_sum_f0_max * 512 + pl->p_bytes;
  const int low_fixed = pl->l_sum_low_max * 512;
  pl->f0_stages = std::min(RC16_MAX_STAGES, (RC16_SMEM_BUDGET - f0_fixed) / RC16_STAGE);

  pl->low_stages = std::min(RC16_MAX_STAGES, (RC16_SMEM_BUDGET - low_fixed) / RC16_STAGE);
  if (f0_fixed > RC16_SMEM_BUDGET || low_fixed > RC16_SMEM_BUDGET || pl->f0_stages < 4 || (pl->n_lr > 0 && pl->low_stages < 4)) return true;
  pl->f0_smem = f0_fixed + pl->f0_stages * RC16_STAGE;
  pl->low_smem = low_fixed + pl->low_stages * RC16_STAGE;
  for (int r = 0; r < pl->n_lr; ++r) {                     // per rate class: R as large as its largest group, the rest is ring
    int lmax = 0;
    for (int b = 0; b < n_bd; ++b) if (!pl->excluded[b]) lmax = std::max(lmax, pl->groups_host[(size_t)b * pl->n_lr + r].l_sum);
    pl->low_geom.r_bytes[r] = lmax * 512;
    pl->low_geom.n_stages[r] = std::min(RC16_MAX_STAGES, (RC16_SMEM_BUDGET - lmax * 512) / RC16_STAGE);
    pl->low_smem = std::max(pl->low_smem, lmax * 512 + pl->low_geom.n_stages[r] * RC16_STAGE);
  }

  // device tables
  std::vector<LowUnit> units;                             // rate-major: all units of a rate have the same tile count
  std::vector<SchedUnit> low_sched;
  for (int r = 0; r < pl->n_lr; ++r) {
    pl->units_per_rate[r] = 0; pl->low_wsum[r] = 0;
    for (int b = 0; b < n_bd; ++b) {
      RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + r];
      if (G.n_slices == 0 || pl->excluded[b]) continue;
      void* q = nullptr;
      if (!plan_alloc(pl, &q, (size_t)G.n_rb * G.q_groups_cap * 4096, true, bytes, err, errlen)) return false;
      G.Q = (__half*)q;
      for (int rb = 0; rb < G.n_rb; ++rb) {
        units.push_back(LowUnit{b * pl->n_lr + r, rb});
        low_sched.push_back(SchedUnit{G.l_sum / 32, (int32_t)pl->low_wsum[r]});
        pl->low_wsum[r] += G.l_sum / 32;
      }
      pl->units_per_rate[r] += G.n_rb;
    }
  }
  // f0 units = combos; cost per tile = ring stages: y chunks of the d == 1 slices + interpolation chunks
  std::vector<SchedUnit> f0_sched;
  pl->f0_wsum = 0;
  for (const F0Combo& cb : pl->combos_host) {
    int w = pl->bd_host[cb.bd].l_sum / 32;
    for (int r = 0; r < pl->n_lr; ++r) {
      if (pl->groups_host[(size_t)cb.bd * pl->n_lr + r].n_slices == 0) continue;
      for (int ch = 0; ch < (pl->up[r].k_win >> 4); ++ch) w += pl->up[r].nn[0][ch] ? 1 : 0;
    }
    f0_sched.push_back(SchedUnit{w, (int32_t)pl->f0_wsum});
    pl->f0_wsum += w;
  }
  pl->low_units = (int)units.size();
  auto upload = [&](void** dst, const void* src, size_t n) -> bool {
    if (!plan_alloc(pl, dst, n, false, bytes, err, errlen)) return false;
    if (n && cudaMemcpy(*dst, src, n, cudaMemcpyHostToDevice) != cudaSuccess) { snprintf(err, errlen, "fp16 plan: table upload failed"); return false; }
    return true;
  };
  if (!upload((void**)&pl->groups_dev, pl->groups_host.data(), pl->groups_host.size() * sizeof(RateGroup))) return false;
  if (!upload((void**)&pl->bd_dev, pl->bd_host.data(), pl->bd_host.size() * sizeof(BdPlan))) return false;
  if (!upload((void**)&pl->combos_dev, pl->combos_host.data(), pl->combos_host.size() * sizeof(F0Combo))) return false;
  if (!upload((void**)&pl->units_dev, units.data(), units.size() * sizeof(LowUnit))) return false;
  if (!upload((void**)&pl->p_dev, pblob.data(), pblob.size() * sizeof(__half))) return false;
  if (!upload((void**)&pl->low_sched_dev, low_sched.data(), low_sched.size() * sizeof(SchedUnit))) return false;
  if (!upload((void**)&pl->f0_sched_dev, f0_sched.data(), f0_sched.size() * sizeof(SchedUnit))) return false;

  cudaError_t e = cudaFuncSetAttribute(f0_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, pl->f0_smem);
  if (e == cudaSuccess && pl->n_lr > 0)
    e = cudaFuncSetAttribute(lowrate_recon_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, pl->low_smem);
  if (e != cudaSuccess) { snprintf(err, errlen, "fp16 plan: cudaFuncSetAttribute failed: %s", cudaGetErrorString(e)); return false; }
  pl->tensor_recon = true;
  return true;
}

bool f16_plan_tensor_recon(const F16Plan* pl) { return pl && pl->tensor_recon; }
void f16_plan_disable_tensor_recon(F16Plan* pl) { if (pl) pl->tensor_recon = false; }
const uint8_t* f16_plan_excluded(const F16Plan* pl) { return (pl && pl->tensor_recon && pl->any_excluded) ? pl->excluded.data() : nullptr; }

int launch_recon_f16(F16Plan* pl, const SliceParams* sp_dev, Peak* partials, int tiles_cap, int max_templates,
                     int c, int64_t k_a, Capture cap, cudaStream_t st, int64_t* launches, cudaEvent_t after_lowrate)
{
  if (pl->low_units > 0) {
    SchedArgs sc;
    memset(&sc, 0, sizeof sc);
    sc.units = pl->low_sched_dev; sc.n_cls = pl->n_lr;
    long long tiles_total = 0;
    for (int r = 0; r < pl->n_lr; ++r) {
      sc.cls_begin[r + 1] = sc.cls_begin[r] + pl->units_per_rate[r];
      sc.n_tiles[r] = (((c >> pl->up[r].log2d) + 2 * kKUp) + 127) / 128;
      sc.cls_base[r + 1] = sc.cls_base[r] + pl->low_wsum[r] * sc.n_tiles[r];
      tiles_total += (long long)sc.n_tiles[r] * pl->units_per_rate[r];
    }
    const int grid = (int)std::min<long long>(pl->n_sm, tiles_total);
    lowrate_recon_kernel<<<grid, LOW_THREADS, pl->low_smem, st>>>(sp_dev, pl->groups_dev, (const LowUnit*)pl->units_dev,
                                                                  sc, pl->low_geom);
    ++*launches;
  }
  if (after_lowrate) cudaEventRecord(after_lowrate, st);
  if (getenv("LLOID_DEBUG_SYNC") && cudaStreamSynchronize(st) != cudaSuccess) { fprintf(stderr, "lloid: lowrate_recon_kernel faulted\n"); return 1; }
  F0Args a;
  memset(&a, 0, sizeof a);
  a.sp = sp_dev; a.bd = pl->bd_dev; a.combos = pl->combos_dev; a.groups = pl->groups_dev;
  a.P = reinterpret_cast<const uint8_t*>(pl->p_dev);
  a.partials = partials; a.cap = cap; a.k_a = k_a;
  a.n_lr = pl->n_lr; a.c = c; a.r_bytes = pl->l_sum_f0_max * 512;
  const int n_combos = (int)pl->combos_host.size();
  const int n_tiles = (c + 127) / 128;
  a.sched.units = pl->f0_sched_dev; a.sched.n_cls = 1;
  a.sched.cls_begin[1] = n_combos; a.sched.n_tiles[0] = n_tiles;
  a.sched.cls_base[1] = pl->f0_wsum * n_tiles;
  // one CTA per SM; a whole number of CTAs per unit (no CTA has to swap R mid-way) only when that leaves at most 3 % of
  // the SMs idle -- 80 units on 148 SMs ran on 80 CTAs before this rule (a 2x step in the time-versus-bins curve)
  int grid = pl->n_sm;
  if (n_combos <= pl->n_sm && n_combos * (pl->n_sm / n_combos) * 100 >= pl->n_sm * 97) grid = n_combos * (pl->n_sm / n_combos);
  grid = (int)std::min<long long>(grid, (long long)n_combos * n_tiles);
  a.tiles_cap = tiles_cap; a.max_templates = max_templates; a.nsy = std::max(2, pl->f0_stages / 3); a.nsq = pl->f0_stages - a.nsy; a.r_bufs = pl->f0_r_bufs; a.p_bytes = pl->p_bytes;
  for (int r = 0; r < kNLowRates; ++r) a.up[r] = pl->up[r];
  for (int r = 0; r < pl->n_lr; ++r)
    for (int v = 0; v < pl->up[r].n_var; ++v)
      for (int ch = 0; ch < (pl->up[r].k_win >> 4); ++ch) {
        const UpRate& U = pl->up[r];
        if (!U.nn[v][ch]) continue;
        QItem& it = a.item[r][v][a.n_items[r][v]++];
        it.idesc = (1u << 4) | ((uint32_t)(U.nn[v][ch] * 8 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);   // idesc_f16(128, N)
        it.b_off = (uint32_t)((U.p_off[v] + 2 * ch * 2048 + U.n0[v][ch] * 128) >> 4);
        it.d_off = (uint32_t)U.n0[v][ch] * 8u;
        it.ch = (uint32_t)ch;
      }
  f0_kernel<<<grid, F0_THREADS, pl->f0_smem, st>>>(a);
  ++*launches;
  const cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) fprintf(stderr, "lloid: f0_kernel launch (grid %d, %d threads, %d B shared, %zu B params): %s\n", grid, F0_THREADS, pl->f0_smem, sizeof a, cudaGetErrorString(e));
  return e == cudaSuccess ? 0 : 1;
}

}  // namespace lloid
