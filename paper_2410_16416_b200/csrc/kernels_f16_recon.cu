// fp16 path (LLOID_F16): A3 reconstruction, A4 upsample + sum and A5 |rho|^2 / windowed maximum on the
// tcgen05 tensor cores (include/lloid.h A3-A5; "matrix multiplication of the orthogonal SNR time
// series with SVD coefficients, and finally up-samples and sums the physical SNR segments").
//
// Round-2 design: CTA PAIRS.  Both kernels run as 2-CTA clusters (one cluster per SM pair, persistent, static
// cost-balanced schedule) and issue cta_group::2 MMAs with M = 256: every CTA owns 128 reconstruction ROWS in their
// natural order (row 2p = cosine, 2p + 1 = sine of template p: 64 templates per CTA, 128 per pair) and HALF of every
// B operand (64 of the 128 time samples of a y tile, 64 of the 128 output columns of a band matrix).  Compared with
// the round-1 kernels (one CTA = 128 templates x 2 accumulators) every per-CTA byte count halves: the stationary R
// (40 KB for L = 160, so L up to 512 and several full-rate slices fit), the y stages, the rho^(d) chunks -- which is
// what buys (a) rings deep enough to cover the memory latency and (b) room to KEEP the rho^(d) windows of consecutive
// tiles in shared memory, so each low-rate sample is fetched once instead of once per overlapping window
// (14 -> 7.75 sixteen-row chunks per tile on BASELINE config 2).
//
//  lowrate_pair_kernel   rho^(d)[i, j] = sum_{slices s at rate d} sum_l R^s[i, l] y^s_l[j]     (d > 1)
//      A = R^s (stationary), B = y^s tiles (ring), D[lane = row, column = low-rate time], four TMEM accumulators of
//      128 columns; epilogue -> fp16 -> Q16, already in the core-matrix layout the f0 kernel consumes as an A operand.
//
//  f0_pair_kernel   rho[i, k] = sum_{d = 1 slices} R^s y^s  +  sum_{d > 1} rho^(d)[i, window(k)] P_d      then A5
//      The interpolation A4 is a tensor-core contraction with the fixed band matrix P_d (16 non-zeros per column),
//      restricted per 16-row chunk to the columns its band touches.  The rho^(d) windows live in per-rate circular
//      buffers: per tile only the rows that entered the window are fetched (one barrier per tile for all rates).
//      Epilogue: a thread owns one ROW (lane); the cosine and sine rows of a template sit in adjacent lanes of one warp
//      and swap half of their columns with one shuffle per column pair; |rho|^2, the running first maximum over a
//      peak-window GRANULE (up to W / 128 tiles) -> ONE 16-byte partial per (template, granule).  The dense f0-rate
//      SNR never leaves TMEM.
//
// Pair plumbing (measured on B200, see tc05.cuh): only the leader CTA issues MMAs; tcgen05.commit multicasts "stage
// free" / "accumulator full" to both CTAs; the peer CTA's loads complete on the peer's own barriers and one relay thread
// per stream forwards "my half has landed" to the leader with a remote arrive.
#include "f16_plan.h"
#include "tc05.cuh"

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <cstdlib>

namespace lloid {

using namespace tc;

constexpr int PK_THREADS = 512;             // 16 warps: 0 PY, 1 IY, 2 PQ, 3 IQ, 4 relay y, 5 relay q, 8-15 epilogue
constexpr int PK_YSTAGE = 8192;             // bytes per y ring stage per CTA: K = 64 x 64 rows
constexpr int PK_NSY_MAX = 16;
constexpr int PK_NACC = 4;                  // accumulator buffers of 128 columns
constexpr int PK_NQB = 4;                   // rho^(d) tile events in flight (barrier slots)
constexpr int PK_QDIST = 2;                 // the rows of tile e are requested when tile e - PK_QDIST has been consumed
constexpr int PK_SMEM_BUDGET = 220 * 1024;  // dynamic; + static (barriers, tables) stays below 227 KB

struct LowUnit { int32_t group, pb; };

struct Ring {                               // stage index + phase parity, advanced without division
  int s; uint32_t ph; int n;
  __device__ __forceinline__ void advance() { if (++s == n) { s = 0; ph ^= 1u; } }
};

// ---- static persistent schedule (SchedArgs in lloid_internal.h), per CLUSTER --------------------------
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

__device__ __forceinline__ int sched_class(const SchedArgs& s, int u)
{
  int c = 0;
  while (c + 1 < s.n_cls && u >= s.cls_begin[c + 1]) ++c;
  return c;
}

// A range boundary inside a unit is moved up to the next granule start (tiles whose absolute index is a multiple of
// gt; gt = 1: no snapping): both ends of every range use the same rule, so the ranges still tile the work.
__device__ __forceinline__ SchedPos sched_snap(const SchedArgs& s, SchedPos p, long long a0, int gt)
{
  if (gt <= 1 || p.t == 0 || p.u >= s.cls_begin[s.n_cls]) return p;
  const int nt = s.n_tiles[sched_class(s, p.u)];
  const int rem = (int)((a0 + p.t) % gt);
  if (rem) p.t += gt - rem;
  if (p.t >= nt) { ++p.u; p.t = 0; }
  return p;
}

// this cluster's range -> rng[0..3] = first unit, first tile, last unit, end tile in the last unit
__device__ __forceinline__ void sched_range(const SchedArgs& s, int cid, int ncl, long long a0, int gt, int* rng)
{
  const long long T = s.cls_base[s.n_cls];
  const SchedPos a = sched_snap(s, sched_locate(s, T * (long long)cid / (long long)ncl), a0, gt);
  const SchedPos b = sched_snap(s, sched_locate(s, T * (long long)(cid + 1) / (long long)ncl), a0, gt);
  rng[0] = a.u; rng[1] = a.t; rng[2] = b.u; rng[3] = b.t;
}

#define FOR_SEGMENTS(u, t0, t1, NT)                                                               \
  for (int u = u_lo; u <= u_hi; ++u)                                                              \
    if (u == u_hi && t_hi == 0) break;                                                            \
    else if (const int t0 = (u == u_lo) ? t_lo : 0, t1 = (u == u_hi) ? t_hi : (NT); t0 >= t1) continue; \
    else

__device__ __forceinline__ void copy_pieces(uint32_t dst, const uint8_t* src, uint32_t bytes, uint32_t bar)
{
  for (uint32_t o = 0; o < bytes; o += 32768u) {
    const uint32_t n = (bytes - o < 32768u) ? bytes - o : 32768u;
    bulk_g2s(dst + o, src + o, n, bar);
  }
}

struct PairBars {
  uint64_t yfull[PK_NSY_MAX], yempty[PK_NSY_MAX];
  uint64_t qfull[PK_NQB], qempty[PK_NQB];
  uint64_t acc_full[PK_NACC], acc_empty[PK_NACC], ybar[PK_NACC];
  uint64_t consts, unit_done;
};

// Barrier counts: a "full" barrier of the leader gets two arrivals (its own producer's arrive.expect_tx and the peer's
// relay), the peer's own copy one.  acc_empty lives in the leader: one arrival per epilogue warp of both CTAs.
__device__ __forceinline__ void pair_setup(PairBars& B, uint32_t* tmem_slot, int nsy, uint32_t rank, int warp, int tid)
{
  if (warp == 0) tmem_alloc2(tmem_slot, 512);
  if (tid == 32) {
    const uint32_t nfull = rank == 0 ? 2u : 1u;
    for (int s = 0; s < nsy; ++s) { mbar_init(smem_u32(&B.yfull[s]), nfull); mbar_init(smem_u32(&B.yempty[s]), 1); }
    for (int s = 0; s < PK_NQB; ++s) { mbar_init(smem_u32(&B.qfull[s]), nfull); mbar_init(smem_u32(&B.qempty[s]), 1); }
    for (int b = 0; b < PK_NACC; ++b) {
      mbar_init(smem_u32(&B.acc_full[b]), 1); mbar_init(smem_u32(&B.acc_empty[b]), 16); mbar_init(smem_u32(&B.ybar[b]), 1);
    }
    mbar_init(smem_u32(&B.consts), nfull);
    mbar_init(smem_u32(&B.unit_done), 1);
    mbar_init_fence();
  }
  fence_before();
  __syncthreads();
  cluster_sync();
  fence_after();
}

__device__ __forceinline__ void pair_teardown(uint32_t tmem, int warp)
{
  fence_before();
  __syncthreads();
  cluster_sync();                           // the peer may still be reading accumulators this CTA's commit announced
  if (warp == 0) tmem_dealloc2(tmem, 512);
}

// producer: wait for the slot to be free, then one bulk copy of `bytes` (<= PK_YSTAGE)
__device__ __forceinline__ void produce(Ring& rg, uint32_t bars_full, uint32_t bars_empty, uint32_t ring_base, const uint8_t* src, uint32_t bytes)
{
  mbar_wait(bars_empty + 8u * rg.s, rg.ph ^ 1u);
  mbar_expect_tx(bars_full + 8u * rg.s, bytes);
  bulk_g2s(ring_base + (uint32_t)rg.s * PK_YSTAGE, src, bytes, bars_full + 8u * rg.s);
  rg.advance();
}

// One y stage (K = ks, a multiple of 16, <= 64) of a reconstruction: D (+)= R[l-groups from a_lo] * stage^T, N = 128.
// a_lo: descriptor of R at this K offset (LBO 2048: 128 rows per l-group); b_lo: descriptor of the stage (LBO 1024: 64 rows)
__device__ __forceinline__ void mma_y_stage(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, int ks, uint32_t& first)
{
  for (int k16 = 0; k16 < (ks >> 4); ++k16) {
    mma2_ss(d_tmem, desc64(a_lo + (uint32_t)k16 * 256u), desc64(b_lo + (uint32_t)k16 * 128u), idesc, first ? 0u : 1u);
    first = 0u;
  }
}

// ------------------------------------------------------------------------------------------------
struct SegSrc {                             // per-role copy of the current unit's operand sources (this CTA's halves)
  const uint8_t* Y[kMaxGroupSlices];        // slice's Y16 base
  const uint8_t* Rsrc[kMaxGroupSlices];     // this CTA's 128-row block of the slice's R16
  int L[kMaxGroupSlices];
  int n;
};

__device__ __forceinline__ void seg_fill(SegSrc& S, const SliceParams* __restrict__ sp, const int32_t* slice, int n, int rb)
{
  S.n = n;
  for (int i = 0; i < n; ++i) {             // one thread
    const SliceParams* P = sp + slice[i];
    const int L = P->L_pad;
    S.Y[i] = reinterpret_cast<const uint8_t*>(P->Y);
    S.Rsrc[i] = reinterpret_cast<const uint8_t*>(P->R16) + (size_t)rb * L * 256;
    S.L[i] = L;
  }
}

// PY role of both kernels: y stages of the unit's slices for tiles [t0, t1) (this CTA's 64-row half of every 128-row
// tile), and the stationary R of the unit.  R goes out after `pre` stages of the new unit are in flight: the ring refills
// while the previous unit drains.  extra/extra_bytes: loaded once with the first R (the f0 kernel's band matrices).
struct PYState { Ring rg; int seg_i; };

__device__ __forceinline__ void py_segment(PYState& st, const SegSrc& sg, PairBars& bars, uint32_t sR_u, uint32_t ring_u,
                                           uint32_t rank, int t0, int t1, uint32_t extra_dst, const uint8_t* extra, uint32_t extra_bytes)
{
  const uint32_t bfull = smem_u32(&bars.yfull[0]), bempty = smem_u32(&bars.yempty[0]);
  int stages_per_tile = 0;
  uint32_t rbytes = 0;
  for (int i = 0; i < sg.n; ++i) { stages_per_tile += (sg.L[i] + 63) >> 6; rbytes += (uint32_t)sg.L[i] * 256u; }
  int pre = (st.seg_i == 0) ? 0 : min(st.rg.n, stages_per_tile);
  bool need_R = true;
  auto load_R = [&]() {
    if (st.seg_i > 0) mbar_wait(smem_u32(&bars.unit_done), (uint32_t)(st.seg_i - 1) & 1u);   // every MMA that reads the old R is complete
    const uint32_t cb = smem_u32(&bars.consts);
    mbar_expect_tx(cb, rbytes + (st.seg_i == 0 ? extra_bytes : 0u));
    uint32_t off = 0;
    for (int i = 0; i < sg.n; ++i) {
      copy_pieces(sR_u + off, sg.Rsrc[i], (uint32_t)sg.L[i] * 256u, cb);
      off += (uint32_t)sg.L[i] * 256u;
    }
    if (st.seg_i == 0 && extra_bytes) copy_pieces(extra_dst, extra, extra_bytes, cb);
    need_R = false;
  };
  if (pre == 0) load_R();
  for (int t = t0; t < t1; ++t)
    for (int i = 0; i < sg.n; ++i) {
      const int L = sg.L[i];
      const uint8_t* src = sg.Y[i] + (size_t)(2 * t + (int)rank) * L * 128;        // 64-row tiles are contiguous in Y16: L / 8 KB each
      for (int k0 = 0; k0 < L; k0 += 64, src += PK_YSTAGE) {
        const int ks = min(64, L - k0);
        produce(st.rg, bfull, bempty, ring_u, src, (uint32_t)ks * 128u);
        if (need_R && --pre == 0) load_R();
      }
    }
  if (need_R) load_R();
  ++st.seg_i;
}

// relay role (peer CTA): forwards the completion of this CTA's y stages and R loads to the leader's barriers
__device__ __forceinline__ void relay_y_segment(Ring& rg, int& seg_i, const SegSrc& sg, PairBars& bars, int t0, int t1)
{
  // consts first (it is requested before or among the first stages of the unit and the leader needs it first)
  mbar_wait(smem_u32(&bars.consts), (uint32_t)seg_i & 1u);
  mbar_arrive_cluster(smem_u32(&bars.consts) & kLeaderMask);
  int stages_per_tile = 0;
  for (int i = 0; i < sg.n; ++i) stages_per_tile += (sg.L[i] + 63) >> 6;
  const uint32_t bfull = smem_u32(&bars.yfull[0]);
  for (int n = (t1 - t0) * stages_per_tile; n > 0; --n) {
    mbar_wait(bfull + 8u * rg.s, rg.ph);
    mbar_arrive_cluster((bfull + 8u * rg.s) & kLeaderMask);
    rg.advance();
  }
  ++seg_i;
}

// ------------------------------------------------------------------------------------------------
struct LowPArgs {
  const SliceParams* sp; const RateGroup* groups; const LowUnit* units;
  int r_bytes, nsy;
  SchedArgs sched;
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PK_THREADS, 1)
lowrate_pair_kernel(const __grid_constant__ LowPArgs a)
{
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) PairBars bars;
  __shared__ uint32_t tmem_slot;
  __shared__ SegSrc seg[3];                             // [0] PY, [1] IY, [2] relay
  __shared__ int s_rng[4];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = cluster_ctarank();
  if (tid == 0) sched_range(a.sched, blockIdx.x >> 1, gridDim.x >> 1, 0, 1, s_rng);
  __syncthreads();
  const int u_lo = s_rng[0], t_lo = s_rng[1], u_hi = s_rng[2], t_hi = s_rng[3];
  if (u_lo == u_hi && t_lo == t_hi) return;             // both CTAs of the cluster take the same decision

  const int nsy = a.nsy;
  pair_setup(bars, &tmem_slot, nsy, rank, warp, tid);
  const uint32_t tmem = tmem_slot;
  const uint32_t sR_u = smem_u32(smem);                 // [l_sum / 8][128 rows][8] fp16
  const uint32_t ring_u = sR_u + (uint32_t)a.r_bytes;

  if (warp == 0) {
    if (elect_one()) {
      PYState st{Ring{0, 0u, nsy}, 0};
      FOR_SEGMENTS(u, t0, t1, a.sched.n_tiles[sched_class(a.sched, u)]) {
        const LowUnit un = a.units[u];
        const RateGroup* G = a.groups + un.group;
        seg_fill(seg[0], a.sp, G->slice, G->n_slices, 2 * un.pb + (int)rank);
        py_segment(st, seg[0], bars, sR_u, ring_u, rank, t0, t1, 0u, nullptr, 0u);
      }
    }
  } else if (warp == 4 && rank == 1) {
    if (elect_one()) {
      Ring rg{0, 0u, nsy};
      int seg_i = 0;
      FOR_SEGMENTS(u, t0, t1, a.sched.n_tiles[sched_class(a.sched, u)]) {
        const LowUnit un = a.units[u];
        const RateGroup* G = a.groups + un.group;
        seg_fill(seg[2], a.sp, G->slice, G->n_slices, 2 * un.pb + (int)rank);
        relay_y_segment(rg, seg_i, seg[2], bars, t0, t1);
      }
    }
  } else if (warp == 1 && rank == 0) {
    // ===== MMA issuer: one elected thread of the leader CTA =====
    if (elect_one()) {
      const uint32_t idesc = idesc_f16_pair(128);
      const uint32_t a_base = desc_lo(sR_u, 2048u), b_base = desc_lo(ring_u, 1024u);
      const uint32_t bfull = smem_u32(&bars.yfull[0]), bempty = smem_u32(&bars.yempty[0]);
      Ring rg{0, 0u, nsy};
      int seg_i = 0;
      uint32_t e = 0;
      FOR_SEGMENTS(u, t0, t1, a.sched.n_tiles[sched_class(a.sched, u)]) {
        const LowUnit un = a.units[u];
        const RateGroup* G = a.groups + un.group;
        seg_fill(seg[1], a.sp, G->slice, G->n_slices, 2 * un.pb);
        mbar_wait_cluster(smem_u32(&bars.consts), (uint32_t)seg_i & 1u);
        fence_after();
        for (int t = t0; t < t1; ++t, ++e) {
          const uint32_t b = e & (PK_NACC - 1), ph = (e >> 2) & 1u;
          mbar_wait_cluster(smem_u32(&bars.acc_empty[b]), ph ^ 1u);
          fence_after();
          const uint32_t d_tmem = tmem + b * 128u;
          uint32_t first = 1u, a_lo = a_base;
          for (int i = 0; i < seg[1].n; ++i) {
            const int L = seg[1].L[i];
            for (int k0 = 0; k0 < L; k0 += 64) {
              const int ks = min(64, L - k0);
              mbar_wait_cluster(bfull + 8u * rg.s, rg.ph);
              fence_after();
              mma_y_stage(d_tmem, a_lo, b_base + (uint32_t)rg.s * (PK_YSTAGE / 16), idesc, ks, first);
              commit2(bempty + 8u * rg.s, 3);
              a_lo += (uint32_t)(ks >> 4) * 256u;
              rg.advance();
            }
          }
          commit2(smem_u32(&bars.acc_full[b]), 3);
        }
        commit2(smem_u32(&bars.unit_done), 3);
        ++seg_i;
      }
    }
  } else if (warp >= 8) {
    // ===== epilogue: thread = row; warps 8-11 columns [0, 64), warps 12-15 columns [64, 128); fp32 -> fp16 -> Q16 =====
    const int q = warp & 3, wg = (warp - 8) >> 2;
    const int row = q * 32 + lane;
    const uint32_t acc_empty_leader = smem_u32(&bars.acc_empty[0]) & kLeaderMask;
    uint32_t e = 0;
    FOR_SEGMENTS(u, t0, t1, a.sched.n_tiles[sched_class(a.sched, u)]) {
      const LowUnit un = a.units[u];
      const RateGroup* Gp = a.groups + un.group;
      const int q_cap = Gp->q_groups_cap;
      __half* __restrict__ Q = Gp->Q + ((size_t)(2 * un.pb + (int)rank) * q_cap * 128 + row) * 8;
      for (int t = t0; t < t1; ++t, ++e) {
        const uint32_t b = e & (PK_NACC - 1), ph = (e >> 2) & 1u;
        mbar_wait(smem_u32(&bars.acc_full[b]), ph);
        fence_after();
        const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + b * 128u + (uint32_t)(64 * wg);
        uint32_t v0[32], v1[32];
        tmem_ld32(taddr, v0);
        tmem_ld32(taddr + 32u, v1);
        tmem_ld_wait();
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(acc_empty_leader + 8u * b);   // the accumulator is in registers: free it first
        const int jg0 = t * 16 + 8 * wg;
#pragma unroll
        for (int gq = 0; gq < 8; ++gq) {
          const uint32_t* v = gq < 4 ? v0 + 8 * gq : v1 + 8 * (gq - 4);
          uint32_t h[4];
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const __half2 p2 = __floats2half2_rn(__uint_as_float(v[2 * x]), __uint_as_float(v[2 * x + 1]));
            h[x] = *reinterpret_cast<const uint32_t*>(&p2);
          }
          if (jg0 + gq < q_cap) *reinterpret_cast<uint4*>(Q + (size_t)(jg0 + gq) * 1024) = make_uint4(h[0], h[1], h[2], h[3]);
        }
      }
    }
  }
  pair_teardown(tmem, warp);
}

// ------------------------------------------------------------------------------------------------
struct F0PArgs {
  const SliceParams* sp; const BdPlan* bd; const F0Combo* combos; const RateGroup* groups;
  const uint8_t* P;                                     // [2][p_bytes]: band-matrix blob of rank 0, of rank 1
  Peak* partials; Capture cap; long long k_a;
  int n_lr, c, r_bytes, p_bytes, q_bytes, nsy, slots_cap, max_templates, gt;
  SchedArgs sched;                                      // units = combos, one class
  PairRate rate[kNLowRates];
};

// chunks (16 low-rate rows) that must be resident before tile t's interpolation: ceil((adv t + adv + 16) / 16)
__device__ __forceinline__ int q_chunks_upto(int adv, int t) { return (adv * t + adv + 16 + 15) >> 4; }

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PK_THREADS, 1)
f0_pair_kernel(const __grid_constant__ F0PArgs a)
{
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) PairBars bars;
  __shared__ uint32_t tmem_slot;
  __shared__ SegSrc seg[3];                             // [0] PY, [1] IY, [2] relay
  __shared__ int s_rng[4];
  __shared__ __align__(16) Peak s_x[2][64];             // epilogue: second column half -> first, per flush parity

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = cluster_ctarank();
  const long long a0 = a.k_a / kTimeTile;               // absolute index of the chunk's tile 0
  if (tid == 0) sched_range(a.sched, blockIdx.x >> 1, gridDim.x >> 1, a0, a.gt, s_rng);
  __syncthreads();
  const int u_lo = s_rng[0], t_lo = s_rng[1], u_hi = s_rng[2], t_hi = s_rng[3];
  if (u_lo == u_hi && t_lo == t_hi) return;
  const int n_tiles = a.sched.n_tiles[0];

  const int nsy = a.nsy, n_lr = a.n_lr;
  pair_setup(bars, &tmem_slot, nsy, rank, warp, tid);
  const uint32_t tmem = tmem_slot;
  const uint32_t sR_u = smem_u32(smem);                 // [l_sum / 8][128 rows][8] fp16
  const uint32_t sP_u = sR_u + (uint32_t)a.r_bytes;     // this rank's band-matrix blocks
  const uint32_t sQ_u = sP_u + (uint32_t)a.p_bytes;     // per-rate circular buffers of 16-row chunks (4 KB each)
  const uint32_t ring_u = sQ_u + (uint32_t)a.q_bytes;   // y ring

  if (warp == 0) {
    // ===== PY: y tiles of the d = 1 slices, R and P =====
    if (elect_one()) {
      PYState st{Ring{0, 0u, nsy}, 0};
      FOR_SEGMENTS(u, t0, t1, n_tiles) {
        const F0Combo cb = a.combos[u];
        const BdPlan* B = a.bd + cb.bd;
        seg_fill(seg[0], a.sp, B->f0_slice, B->n_f0, 2 * cb.rb + (int)rank);
        py_segment(st, seg[0], bars, sR_u, ring_u, rank, t0, t1, sP_u, a.P + (size_t)rank * a.p_bytes, (uint32_t)a.p_bytes);
      }
    }
  } else if (warp == 4 && rank == 1) {
    if (elect_one()) {
      Ring rg{0, 0u, nsy};
      int seg_i = 0;
      FOR_SEGMENTS(u, t0, t1, n_tiles) {
        const F0Combo cb = a.combos[u];
        const BdPlan* B = a.bd + cb.bd;
        seg_fill(seg[2], a.sp, B->f0_slice, B->n_f0, 2 * cb.rb + (int)rank);
        relay_y_segment(rg, seg_i, seg[2], bars, t0, t1);
      }
    }
  } else if (warp == 2) {
    // ===== PQ: the rows of every rate's rho^(d) window that tile e needs and tile e - 1 did not have =====
    if (elect_one()) {
      uint32_t e = 0;
      FOR_SEGMENTS(u, t0, t1, n_tiles) {
        const F0Combo cb = a.combos[u];
        const uint8_t* qsrc[kNLowRates];
        for (int r = 0; r < n_lr; ++r) {
          const RateGroup* G = a.groups + cb.bd * n_lr + r;
          qsrc[r] = (G->n_slices > 0) ? reinterpret_cast<const uint8_t*>(G->Q) + (size_t)(2 * cb.rb + (int)rank) * G->q_groups_cap * 2048 : nullptr;
        }
        for (int t = t0; t < t1; ++t, ++e) {
          // a unit's first tile fetches whole windows into slots other tiles may still be reading: drain first
          if (t == t0) { if (e > 0) mbar_wait(smem_u32(&bars.qempty[(e - 1) & (PK_NQB - 1)]), ((e - 1) >> 2) & 1u); }
          else if (e >= PK_QDIST) mbar_wait(smem_u32(&bars.qempty[(e - PK_QDIST) & (PK_NQB - 1)]), ((e - PK_QDIST) >> 2) & 1u);
          const uint32_t fb = smem_u32(&bars.qfull[e & (PK_NQB - 1)]);
          uint32_t total = 0;
          for (int r = 0; r < n_lr; ++r) {
            if (!qsrc[r]) continue;
            const int adv = a.rate[r].adv;
            const int c_lo = (t == t0) ? (adv * t) >> 4 : q_chunks_upto(adv, t - 1);
            total += (uint32_t)(q_chunks_upto(adv, t) - c_lo) * 4096u;
          }
          mbar_expect_tx(fb, total);                    // total == 0: a plain arrival
          for (int r = 0; r < n_lr; ++r) {
            if (!qsrc[r]) continue;
            const int adv = a.rate[r].adv, cap = a.rate[r].cap_chunks;
            const int c_lo = (t == t0) ? (adv * t) >> 4 : q_chunks_upto(adv, t - 1);
            const int c_hi = q_chunks_upto(adv, t);
            if (c_hi <= c_lo) continue;
            const uint32_t base = sQ_u + (uint32_t)a.rate[r].ring_off;
            const int s0 = c_lo % cap;
            const int n1 = min(c_hi - c_lo, cap - s0);
            copy_pieces(base + (uint32_t)s0 * 4096u, qsrc[r] + (size_t)c_lo * 4096, (uint32_t)n1 * 4096u, fb);
            if (c_hi - c_lo > n1) copy_pieces(base, qsrc[r] + (size_t)(c_lo + n1) * 4096, (uint32_t)(c_hi - c_lo - n1) * 4096u, fb);
          }
        }
      }
    }
  } else if (warp == 5 && rank == 1) {
    // ===== relay of the rho^(d) tile events =====
    if (elect_one()) {
      uint32_t e = 0;
      FOR_SEGMENTS(u, t0, t1, n_tiles) {
        for (int t = t0; t < t1; ++t, ++e) {
          const uint32_t fb = smem_u32(&bars.qfull[e & (PK_NQB - 1)]);
          mbar_wait(fb, (e >> 2) & 1u);
          mbar_arrive_cluster(fb & kLeaderMask);
        }
      }
    }
  } else if (warp == 1 && rank == 0) {
    // ===== IY: MMAs of the d = 1 slices =====
    if (elect_one()) {
      const uint32_t idesc = idesc_f16_pair(128);
      const uint32_t a_base = desc_lo(sR_u, 2048u), b_base = desc_lo(ring_u, 1024u);
      const uint32_t bfull = smem_u32(&bars.yfull[0]), bempty = smem_u32(&bars.yempty[0]);
      Ring rg{0, 0u, nsy};
      int seg_i = 0;
      uint32_t e = 0;
      FOR_SEGMENTS(u, t0, t1, n_tiles) {
        const F0Combo cb = a.combos[u];
        const BdPlan* B = a.bd + cb.bd;
        seg_fill(seg[1], a.sp, B->f0_slice, B->n_f0, 2 * cb.rb);
        mbar_wait_cluster(smem_u32(&bars.consts), (uint32_t)seg_i & 1u);
        fence_after();
        for (int t = t0; t < t1; ++t, ++e) {
          const uint32_t b = e & (PK_NACC - 1), ph = (e >> 2) & 1u;
          mbar_wait_cluster(smem_u32(&bars.acc_empty[b]), ph ^ 1u);
          fence_after();
          const uint32_t d_tmem = tmem + b * 128u;
          uint32_t first = 1u, a_lo = a_base;
          for (int i = 0; i < seg[1].n; ++i) {
            const int L = seg[1].L[i];
            for (int k0 = 0; k0 < L; k0 += 64) {
              const int ks = min(64, L - k0);
              mbar_wait_cluster(bfull + 8u * rg.s, rg.ph);
              fence_after();
              mma_y_stage(d_tmem, a_lo, b_base + (uint32_t)rg.s * (PK_YSTAGE / 16), idesc, ks, first);
              commit2(bempty + 8u * rg.s, 3);
              a_lo += (uint32_t)(ks >> 4) * 256u;
              rg.advance();
            }
          }
          commit2(smem_u32(&bars.ybar[b]), 1);
        }
        ++seg_i;
      }
    }
  } else if (warp == 3 && rank == 0) {
    // ===== IQ: interpolation MMAs (A4), after the tile's y part is complete =====
    if (elect_one()) {
      const uint32_t p_base = sP_u >> 4;
      uint32_t e = 0;
      FOR_SEGMENTS(u, t0, t1, n_tiles) {
        const F0Combo cb = a.combos[u];
        uint32_t present = 0;
        for (int r = 0; r < n_lr; ++r) if (a.groups[cb.bd * n_lr + r].n_slices > 0) present |= 1u << r;
        for (int t = t0; t < t1; ++t, ++e) {
          const uint32_t b = e & (PK_NACC - 1), ph = (e >> 2) & 1u;
          mbar_wait(smem_u32(&bars.ybar[b]), ph);
          mbar_wait_cluster(smem_u32(&bars.qfull[e & (PK_NQB - 1)]), ph);
          fence_after();
          const uint32_t d_tmem = tmem + b * 128u;
          for (int r = 0; r < n_lr; ++r) {
            if (!(present >> r & 1u)) continue;
            const PairRate& R = a.rate[r];
            const int v = (R.adv >= 16) ? 0 : ((R.adv * t) & 15) / R.adv;
            const int s0 = ((R.adv * t) >> 4) % R.cap_chunks;
            const uint32_t qa = desc_lo(sQ_u + (uint32_t)R.ring_off, 2048u);
            const int n_it = R.n_items[v];
            for (int k = 0; k < n_it; ++k) {
              const PairItem it = R.item[v][k];
              int s = s0 + (int)it.ch; if (s >= R.cap_chunks) s -= R.cap_chunks;
              mma2_ss(d_tmem + it.d_col, desc64(qa + (uint32_t)s * 256u), desc64(p_base + it.p_lo), it.idesc, 1u);
            }
          }
          commit2(smem_u32(&bars.qempty[e & (PK_NQB - 1)]), 3);
          commit2(smem_u32(&bars.acc_full[b]), 3);
        }
        commit2(smem_u32(&bars.unit_done), 3);
      }
    }
  } else if (warp >= 8) {
    // ===== epilogue: thread = row (lane); lanes 2i / 2i + 1 of a warp hold the cosine / sine row of one template =====
    const int q = warp & 3, wg = (warp - 8) >> 2;
    const int row = q * 32 + lane;
    const int part = lane & 1;
    const uint32_t acc_empty_leader = smem_u32(&bars.acc_empty[0]) & kLeaderMask;
    uint32_t e = 0, flush_i = 0;
    FOR_SEGMENTS(u, t0, t1, n_tiles) {
      const F0Combo cb = a.combos[u];
      const int n_templates = a.bd[cb.bd].n_templates;
      const int grow = (2 * cb.rb + (int)rank) * 128 + row;             // reconstruction row i = 2 p + part
      const int p = grow >> 1;
      const bool capture = a.cap.snr != nullptr && a.cap.bd == cb.bd && grow < a.cap.rows;
      // running first maximum of this thread's columns over the current granule
      float bq = -1.f, bmine = 0.f, brecv = 0.f;
      int bk = 0;
      for (int t = t0; t < t1; ++t, ++e) {
        const uint32_t b = e & (PK_NACC - 1), ph = (e >> 2) & 1u;
        mbar_wait(smem_u32(&bars.acc_full[b]), ph);
        fence_after();
        const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + b * 128u + (uint32_t)(64 * wg);
        uint32_t lo[32], hi[32];                        // columns 64 wg + [0, 32) and + [32, 64) of this row
        tmem_ld32(taddr, lo);
        tmem_ld32(taddr + 32u, hi);
        tmem_ld_wait();
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(acc_empty_leader + 8u * b);   // the tile is in registers: free the accumulator
        const int kap0 = t * 128;
        const int valid = min(128, a.c - kap0);
        if (capture) {
#pragma unroll
          for (int j = 0; j < 64; ++j) {
            const int col = 64 * wg + j;
            const long long k = a.k_a + kap0 + col;
            if (col < valid && k >= a.cap.k_begin && k < a.cap.k_begin + a.cap.n)
              a.cap.snr[(size_t)grow * a.cap.n + (k - a.cap.k_begin)] = __uint_as_float(j < 32 ? lo[j] : hi[j - 32]);
          }
        }
        // even lanes (cosine row) take columns [0, 32) of the 64, odd lanes (sine row) [32, 64): one shuffle per column
        // brings the partner row's value of the SAME column
        const int cbase = 64 * wg + 32 * part;
        float q4[4] = {-1.f, -1.f, -1.f, -1.f}, m4[4] = {0.f, 0.f, 0.f, 0.f}, r4[4] = {0.f, 0.f, 0.f, 0.f};
        int k4[4] = {0, 0, 0, 0};
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const float send = __uint_as_float(part ? lo[j] : hi[j]);
          const float mine = __uint_as_float(part ? hi[j] : lo[j]);
          const float recv = __shfl_xor_sync(0xffffffffu, send, 1);
          const float qq = fmaf(mine, mine, recv * recv);
          if (cbase + j < valid && qq > q4[j & 3]) { q4[j & 3] = qq; k4[j & 3] = cbase + j; m4[j & 3] = mine; r4[j & 3] = recv; }
        }
        float tq = q4[0], tm = m4[0], tr = r4[0];
        int tk = k4[0];
#pragma unroll
        for (int m = 1; m < 4; ++m)
          if (q4[m] > tq || (q4[m] == tq && k4[m] < tk)) { tq = q4[m]; tk = k4[m]; tm = m4[m]; tr = r4[m]; }
        if (tq > bq) { bq = tq; bk = kap0 + tk; bmine = tm; brecv = tr; }      // later tiles never win ties
        // granule end: merge the four partial maxima of a template (two lanes x two column halves), write one record
        const long long at = a0 + t;
        if (t + 1 == t1 || (at + 1) % a.gt == 0) {
          // partner lane: the odd lane's columns are later, so the even lane wins ties
          const float oq = __shfl_xor_sync(0xffffffffu, bq, 1), om = __shfl_xor_sync(0xffffffffu, bmine, 1), orv = __shfl_xor_sync(0xffffffffu, brecv, 1);
          const int ok = __shfl_xor_sync(0xffffffffu, bk, 1);
          float re = part ? brecv : bmine, im = part ? bmine : brecv;          // this thread's best as (re, im)
          const float ore = part ? om : orv, oim = part ? orv : om;            // partner's best (its part is the other one)
          if (oq > bq || (oq == bq && ok < bk)) { bq = oq; bk = ok; re = ore; im = oim; }
          const int fp = flush_i & 1;
          if (wg == 1 && part == 0) { Peak pk; pk.q = bq; pk.kappa = bk; pk.re = re; pk.im = im; s_x[fp][row >> 1] = pk; }
          asm volatile("bar.sync 2, 256;" ::: "memory");
          if (wg == 0 && part == 0) {
            const Peak o = s_x[fp][row >> 1];
            if (o.q > bq) { bq = o.q; bk = o.kappa; re = o.re; im = o.im; }    // its columns are later: ties stay here
            if (p < n_templates) {
              const int gi = (int)(at / a.gt - a0 / a.gt);
              Peak pk; pk.q = bq; pk.kappa = bk; pk.re = re; pk.im = im;
              a.partials[((size_t)cb.bd * a.slots_cap + gi) * a.max_templates + p] = pk;
            }
          }
          ++flush_i;
          bq = -1.f; bk = 0; bmine = 0.f; brecv = 0.f;
        }
      }
    }
  }
  pair_teardown(tmem, warp);
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

inline int chunks_upto(int adv, int t) { return (adv * t + adv + 16 + 15) >> 4; }

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
  for (int l2 = 1; l2 < kMaxRates; ++l2) { lr_of[l2] = -1; if (have[l2]) { lr_of[l2] = pl->n_lr; pl->rate[pl->n_lr].log2d = l2; ++pl->n_lr; } }

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
    B.n_rb = (B.n_templates + kTplBlock - 1) / kTplBlock;              // pair blocks of 128 templates
    for (int r = 0; r < pl->n_lr; ++r) {
      RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + r];
      memset(&G, 0, sizeof G);
      G.log2d = pl->rate[r].log2d; G.n_rb = B.n_rb;
      G.q_groups_cap = (((chunk_cap >> G.log2d) + 2 * kKUp + 127) / 128) * 16 + 16;
    }
    for (int s = 0; s < bp_host[b].n_slices; ++s) {
      const int idx = bp_host[b].first_slice + s;
      const SliceParams& P = sp_host[idx];
      if (P.rows_pad != B.n_rb * 2 * kTplBlock || P.L_pad % 16) { ok = false; break; }
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

  // Band matrices P_d (A4), one block per (rate, variant, 16-row chunk of the window):
  //   c[kl] = sum_rw Q[16 floor(adv t / 16) + rw] P[rw, kl],  mis = adv t mod 16 (variant = mis / adv),
  //   P[rw, kl] = w_phi[i], i = mis + floor(kl / d) + K_up - rw in [-K_up, K_up), phi = kl mod d.
  // A block keeps the nn columns [n0, n0 + nn) its band touches; rank 0 stores columns [n0, n0 + nn / 2), rank 1 the
  // rest (B operand of a cta_group::2 MMA), each as [2 row groups][nn / 2 columns][8 rows] fp16.
  std::vector<__half> pblob[2];
  int q_bytes = 0;
  for (int r = 0; r < pl->n_lr; ++r) {
    PairRate& U = pl->rate[r];
    const int l2 = U.log2d, d = 1 << l2;
    if (!up_w || !up_w[l2]) return true;
    const double* w = up_w[l2];
    U.adv = 128 >> l2;
    U.n_var = U.adv >= 16 ? 1 : 16 / U.adv;
    if (U.n_var > 4) return true;
    // circular buffer: every chunk that tile t - PK_QDIST + 1 .. t may still read, while tile t's rows arrive
    int cap = 0;
    for (int t = 0; t < 64; ++t) cap = std::max(cap, chunks_upto(U.adv, t) - ((U.adv * std::max(t - PK_QDIST + 1, 0)) >> 4));
    U.cap_chunks = cap;
    U.ring_off = q_bytes;
    q_bytes += cap * 4096;
    for (int v = 0; v < 4; ++v) U.n_items[v] = 0;
    for (int v = 0; v < U.n_var; ++v) {
      const int mis = v * U.adv;
      const int nch = (mis + U.adv + 2 * kKUp + 15) / 16;
      if (nch > 5) return true;
      for (int ch = 0; ch < nch; ++ch) {
        int cmin = 1 << 30, cmax = -1;
        for (int rr = 0; rr < 16; ++rr)
          for (int kl = 0; kl < 128; ++kl) {
            const int i = mis + kl / d + kKUp - (16 * ch + rr);
            if (i < -kKUp || i >= kKUp) continue;
            cmin = std::min(cmin, kl); cmax = std::max(cmax, kl);
          }
        if (cmax < 0) continue;
        int n0 = cmin / 8 * 8;
        const int nn = (cmax + 1 - n0 + 15) / 16 * 16;
        if (n0 + nn > 128) n0 = 128 - nn;
        const int half = nn / 2;
        const size_t base = pblob[0].size();
        for (int c = 0; c < 2; ++c) pblob[c].resize(base + (size_t)16 * half, __float2half(0.f));
        for (int rr = 0; rr < 16; ++rr)
          for (int j = 0; j < nn; ++j) {
            const int kl = n0 + j;
            const int i = mis + kl / d + kKUp - (16 * ch + rr);
            if (i < -kKUp || i >= kKUp) continue;
            pblob[j / half][base + ((size_t)(rr >> 3) * half + (j % half)) * 8 + (rr & 7)] = __float2half_rn((float)w[(size_t)(i + kKUp) * d + kl % d]);
          }
        PairItem& it = U.item[v][U.n_items[v]++];
        it.idesc = (1u << 4) | ((uint32_t)(nn >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
        it.p_lo = (uint32_t)((base * sizeof(__half)) >> 4) | ((uint32_t)half << 16);     // LBO = half * 16 bytes
        it.d_col = (uint32_t)n0;
        it.ch = (uint32_t)ch;
      }
    }
  }
  pl->p_bytes = (int)((pblob[0].size() * sizeof(__half) + 127) / 128 * 128);
  pl->q_bytes = q_bytes;

  // per-(bin, detector) shared-memory limits: stationary R (this CTA's 128 rows) + P + windows + >= 3 y stages
  {
    const int lim_f0 = (PK_SMEM_BUDGET - pl->p_bytes - pl->q_bytes - 3 * PK_YSTAGE) / 256;
    const int lim_low = (PK_SMEM_BUDGET - 3 * PK_YSTAGE) / 256;
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
  const int f0_fixed = pl->l_sum_f0_max * 256 + pl->p_bytes + pl->q_bytes;
  const int low_fixed = pl->l_sum_low_max * 256;
  pl->f0_stages = std::min(PK_NSY_MAX, (PK_SMEM_BUDGET - f0_fixed) / PK_YSTAGE);
  pl->low_stages = std::min(PK_NSY_MAX, (PK_SMEM_BUDGET - low_fixed) / PK_YSTAGE);
  pl->f0_smem = f0_fixed + pl->f0_stages * PK_YSTAGE;
  pl->low_smem = low_fixed + pl->low_stages * PK_YSTAGE;

  // device tables
  std::vector<LowUnit> units;                             // rate-major: all units of a rate have the same tile count
  std::vector<SchedUnit> low_sched;
  for (int r = 0; r < pl->n_lr; ++r) {
    pl->units_per_rate[r] = 0; pl->low_wsum[r] = 0;
    for (int b = 0; b < n_bd; ++b) {
      RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + r];
      if (G.n_slices == 0 || pl->excluded[b]) continue;
      void* q = nullptr;
      if (!plan_alloc(pl, &q, (size_t)G.n_rb * 2 * G.q_groups_cap * 2048, true, bytes, err, errlen)) return false;
      G.Q = (__half*)q;
      for (int rb = 0; rb < G.n_rb; ++rb) {
        units.push_back(LowUnit{b * pl->n_lr + r, rb});
        low_sched.push_back(SchedUnit{G.l_sum / 16, (int32_t)pl->low_wsum[r]});
        pl->low_wsum[r] += G.l_sum / 16;
      }
      pl->units_per_rate[r] += G.n_rb;
    }
  }
  // f0 units = combos; cost per tile = MMAs: K / 16 of the d == 1 slices + interpolation chunks
  std::vector<SchedUnit> f0_sched;
  pl->f0_wsum = 0;
  for (const F0Combo& cb : pl->combos_host) {
    int w = pl->bd_host[cb.bd].l_sum / 16;
    for (int r = 0; r < pl->n_lr; ++r) {
      if (pl->groups_host[(size_t)cb.bd * pl->n_lr + r].n_slices == 0) continue;
      w += pl->rate[r].n_items[0];
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
  {
    std::vector<uint8_t> both((size_t)2 * pl->p_bytes + 16, 0);
    for (int c = 0; c < 2; ++c) memcpy(both.data() + (size_t)c * pl->p_bytes, pblob[c].data(), pblob[c].size() * sizeof(__half));
    if (!upload((void**)&pl->p_dev, both.data(), both.size())) return false;
  }
  if (!upload((void**)&pl->low_sched_dev, low_sched.data(), low_sched.size() * sizeof(SchedUnit))) return false;
  if (!upload((void**)&pl->f0_sched_dev, f0_sched.data(), f0_sched.size() * sizeof(SchedUnit))) return false;

  // opt-in shared memory: the architecture maximum, for every kernel of this file, on this device (never lowered
  // by a later, smaller bank)
  cudaError_t e = set_max_dyn_smem(f0_pair_kernel);
  if (e == cudaSuccess) e = set_max_dyn_smem(lowrate_pair_kernel);
  if (e != cudaSuccess) { snprintf(err, errlen, "fp16 plan: cudaFuncSetAttribute failed: %s", cudaGetErrorString(e)); return false; }
  pl->tensor_recon = true;
  return true;
}

bool f16_plan_tensor_recon(const F16Plan* pl) { return pl && pl->tensor_recon; }
void f16_plan_disable_tensor_recon(F16Plan* pl) { if (pl) pl->tensor_recon = false; }
const uint8_t* f16_plan_excluded(const F16Plan* pl) { return (pl && pl->tensor_recon && pl->any_excluded) ? pl->excluded.data() : nullptr; }

int f16_granule_tiles(int peak_window)
{
  int gt = peak_window / kTimeTile;
  while (gt > 32 && gt % 2 == 0) gt /= 2;
  return gt < 1 ? 1 : gt;
}

int launch_recon_f16(F16Plan* pl, const SliceParams* sp_dev, Peak* partials, int slots_cap, int max_templates,
                     int c, int64_t k_a, int gt, Capture cap, cudaStream_t st, int64_t* launches, cudaEvent_t after_lowrate)
{
  const int n_clusters = std::max(1, pl->n_sm / 2);
  if (pl->low_units > 0) {
    LowPArgs la;
    memset(&la, 0, sizeof la);
    la.sp = sp_dev; la.groups = pl->groups_dev; la.units = (const LowUnit*)pl->units_dev;
    la.r_bytes = pl->l_sum_low_max * 256; la.nsy = pl->low_stages;
    SchedArgs& sc = la.sched;
    sc.units = pl->low_sched_dev; sc.n_cls = pl->n_lr;
    long long tiles_total = 0;
    for (int r = 0; r < pl->n_lr; ++r) {
      sc.cls_begin[r + 1] = sc.cls_begin[r] + pl->units_per_rate[r];
      sc.n_tiles[r] = (((c >> pl->rate[r].log2d) + 2 * kKUp) + 127) / 128;
      sc.cls_base[r + 1] = sc.cls_base[r] + pl->low_wsum[r] * sc.n_tiles[r];
      tiles_total += (long long)sc.n_tiles[r] * pl->units_per_rate[r];
    }
    const int grid = 2 * (int)std::min<long long>(n_clusters, tiles_total);
    lowrate_pair_kernel<<<grid, PK_THREADS, pl->low_smem, st>>>(la);
    ++*launches;
  }
  if (after_lowrate) cudaEventRecord(after_lowrate, st);
  if (getenv("LLOID_DEBUG_SYNC") && cudaStreamSynchronize(st) != cudaSuccess) { fprintf(stderr, "lloid: lowrate_pair_kernel faulted\n"); return 1; }
  F0PArgs a;
  memset(&a, 0, sizeof a);
  a.sp = sp_dev; a.bd = pl->bd_dev; a.combos = pl->combos_dev; a.groups = pl->groups_dev;
  a.P = reinterpret_cast<const uint8_t*>(pl->p_dev);
  a.partials = partials; a.cap = cap; a.k_a = k_a;
  a.n_lr = pl->n_lr; a.c = c; a.r_bytes = pl->l_sum_f0_max * 256; a.p_bytes = pl->p_bytes; a.q_bytes = pl->q_bytes;
  a.nsy = pl->f0_stages; a.slots_cap = slots_cap; a.max_templates = max_templates; a.gt = gt;
  const int n_combos = (int)pl->combos_host.size();
  const int n_tiles = (c + 127) / 128;
  a.sched.units = pl->f0_sched_dev; a.sched.n_cls = 1;
  a.sched.cls_begin[1] = n_combos; a.sched.n_tiles[0] = n_tiles;
  a.sched.cls_base[1] = pl->f0_wsum * n_tiles;
  for (int r = 0; r < kNLowRates; ++r) a.rate[r] = pl->rate[r];
  const int grid = 2 * (int)std::min<long long>(n_clusters, (long long)n_combos * n_tiles);
  f0_pair_kernel<<<grid, PK_THREADS, pl->f0_smem, st>>>(a);
  ++*launches;
  const cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) fprintf(stderr, "lloid: f0_pair_kernel launch (grid %d, %d threads, %d B shared, %zu B params): %s\n", grid, PK_THREADS, pl->f0_smem, sizeof a, cudaGetErrorString(e));
  return e == cudaSuccess ? 0 : 1;
}

}  // namespace lloid
