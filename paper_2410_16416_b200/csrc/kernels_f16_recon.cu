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

constexpr int PK_THREADS = 512;             // 16 warps (4 per scheduler: 128 registers per thread): 0 PY, 1 IY (leader), 2 PQ0, 3 IQ0 (leader),
                                            // 4 relay y (peer), 5 IQ1 (leader) / relay q (peer), 6 PQ1, 7 L2 prefetcher, 8-15 epilogue
constexpr int PK_NSY_MAX = 16;
constexpr int PK_NACC_MAX = 4;              // accumulator buffers of 128 columns: 4 with R in shared memory, 2 with R in TMEM
constexpr int PK_ACOL = 256;                // R in TMEM: columns [256, 256 + K / 2) beside two accumulators
constexpr int PK_KMAX = 512;                // ... so a unit's summed L_pad is at most 512 there
// Both kernels exist in two variants (template parameter RT).  RT = false: the unit's stationary R (128 rows x K per CTA) sits
// in shared memory and every y MMA reads both operands from there -- the fastest variant on BASELINE config 2, but R, the band
// matrices, the rho^(d) windows and the y ring must share 218 KB, which holds K <= ~320.  RT = true: the epilogue warps copy R
// into TMEM once per unit and the y MMAs take A from TMEM (tcgen05.mma [d], [a], b-desc): K up to 512 (BASELINE config 4:
// L up to 300 on the full-rate slice), half the shared-memory operand traffic, but only two accumulators.  The plan picks
// RT = true only when some (bin, detector) needs it.
template <bool RT> struct Acc { static constexpr uint32_t N = RT ? 2u : 4u; };
constexpr int PK_NQB = 4;                   // rho^(d) tile events in flight (barrier slots)
constexpr int PK_QDIST = 2;                 // the rows of tile e are requested when tile e - PK_QDIST has been consumed
constexpr int PK_QPF = 4;                   // L2 prefetch distance of the rho^(d) rows, in tiles
constexpr int PK_YPF = 4;                   // L2 prefetch distance of the y tiles, in tiles
constexpr int PK_SMEM_BUDGET = 218 * 1024;  // dynamic; + static (barriers, tables) stays below 227 KB

struct LowUnit { int32_t group, pb; };

// Role trace (scratch builds with -DLLOID_TRACE_BUILD and LLOID_TRACE=1): cycles each single-thread role of cluster 0
// spends waiting on each of its barriers and in total, accumulated over the launches; read back with lloid_debug_trace.
__device__ long long g_trace[2][8][8];
#ifdef LLOID_TRACE_BUILD
__constant__ int g_exp;                      // scratch knock-outs: 1 no interpolation MMAs, 2 no y MMAs (f0), 4 no epilogue arithmetic (f0)
#endif      // [kernel: 0 low, 1 f0][role][0..5 wait categories, 6 total, 7 tiles]
#ifdef LLOID_TRACE_BUILD
#define TWAIT(cat, bar, ph)                                                                       \
  do { if (trace) { const long long t_ = clock64(); mbar_wait(bar, ph); tw[cat] += clock64() - t_; } else mbar_wait(bar, ph); } while (0)
#define TRACE_BEGIN() const bool trace = a.trace && (blockIdx.x >> 1) == 0; long long tw[6] = {0, 0, 0, 0, 0, 0}; const long long tbeg = trace ? clock64() : 0
#define TSPAN_BEGIN() const long long ts_ = trace ? clock64() : 0
#define TSPAN_END(cat) do { if (trace) tw[cat] += clock64() - ts_; } while (0)
#define TRACE_END(kern, role, ntiles) do { if (trace) { for (int i_ = 0; i_ < 6; ++i_) g_trace[kern][role][i_] += tw[i_]; g_trace[kern][role][6] += clock64() - tbeg; g_trace[kern][role][7] += (ntiles); } } while (0)
#else
#define TWAIT(cat, bar, ph) mbar_wait(bar, ph)
#define TRACE_BEGIN() constexpr bool trace = false; long long* const tw = nullptr; (void)trace; (void)tw
#define TSPAN_BEGIN() do { } while (0)
#define TSPAN_END(cat) do { } while (0)
#define TRACE_END(kern, role, ntiles) do { (void)(ntiles); } while (0)
#endif

// A single thread retires roughly one dependent instruction per 5-7 cycles (measured: a loop around one MMA with ~15
// instructions of address arithmetic issues an MMA every 99 cycles; with the MMAs and the copies knocked out the handshake
// skeleton of the first version of this file still took longer than the MMAs).  The role loops below are written for
// instruction count -- y stages carry up to K = 128, barrier addresses are hoisted, the interpolation MMAs read their
// operands from a table in the kernel parameters -- and the two MMA-issuing roles exist TWICE, one thread for the even
// tiles and one for the odd tiles (different accumulators, so the pipe needs no ordering between them).
struct YRing {                              // y ring position: slot index + phase parity (+ tiles started: PY only)
  uint32_t s, ph, n, tiles = 0;
  __device__ __forceinline__ void advance() { if (++s == n) { s = 0; ph ^= 1u; } }
  __device__ __forceinline__ void skip(uint32_t k) { s += k; while (s >= n) { s -= n; ph ^= 1u; } }
};

// ---- f0 kernel schedule ------------------------------------------------------------------------------------------
// The flattened work sequence is ordered by (bin, detector), then by time BLOCKS of gb tiles (aligned to absolute tile
// indices), then by template block, then by tile; cluster i takes the cost range [T i / G, T (i + 1) / G) of it, its ends
// moved up to granule starts.  With a block of one cluster's share (launch_recon_f16) cluster i works on about the i-th
// (time block, template block) cell: the clusters that reconstruct the template blocks of one time block from the same y
// tiles run side by side and all but one of them find a y tile in L2.
// n_pb > 0 selects the order (time block, template block, (bin, detector), tile) instead -- meant for banks with many
// (bin, detector) pairs per chunk, where a cluster walks the template blocks of a pair one after the other and y comes
// from DRAM every time (config 4: 3 GB of reads per launch for 1 GB of operands).  It needs the same number of template
// blocks for every pair.  Measured (LLOID_F0_ORDER_PB): clusters G / n_pb apart do not stay in step; DRAM reads 3.5 -> 3.0
// GB on config 4, 0.88 -> 1.07 GB on config 2, no gain in time.  Kept, off.
struct F0Sched {
  const SchedBd* bds;                       // tensor-path (bin, detector) pairs, in order
  int n_bds, n_tiles, gb, gt;
  int n_pb;                                 // template blocks of every entry if they all agree, else 0
  long long total;                          // sum of n_pb * w
  long long a0;                             // absolute index of the chunk's tile 0
};
struct F0Pos { int ib, lo, hi, pb, t; };    // index into bds, block [lo, hi) in chunk tiles, template block, tile

__device__ __forceinline__ int f0_first_block_end(const F0Sched& S) { return min(S.n_tiles, S.gb - (int)(S.a0 % S.gb)); }

__device__ __forceinline__ void f0_next_cell(const F0Sched& S, F0Pos& p)      // next cell in order
{
  if (S.n_pb) {                             // (time block, template block, bd): past the end lo == n_tiles
    if (++p.ib < S.n_bds) { p.t = p.lo; return; }
    p.ib = 0;
    if (++p.pb < S.n_pb) { p.t = p.lo; return; }
    p.pb = 0; p.lo = p.hi; p.hi = min(S.n_tiles, p.hi + S.gb); p.t = p.lo;
    return;
  }
  if (++p.pb < S.bds[p.ib].n_pb) { p.t = p.lo; return; }
  p.pb = 0; p.lo = p.hi; p.hi = min(S.n_tiles, p.hi + S.gb); p.t = p.lo;
  if (p.lo >= S.n_tiles) { ++p.ib; p.lo = 0; p.hi = f0_first_block_end(S); p.t = 0; }
}

__device__ __forceinline__ void f0_granule_up(const F0Sched& S, F0Pos& p)      // move up to the next granule start
{
  if (p.t > p.lo) {
    const int r = (int)((S.a0 + p.t) % S.gt);
    if (r) p.t += S.gt - r;
    if (p.t >= p.hi) f0_next_cell(S, p);
  }
}

__device__ __forceinline__ F0Pos f0_locate(const F0Sched& S, long long pos)
{
  F0Pos p;
  const long long nt = S.n_tiles;
  if (S.n_pb) {
    if (pos >= S.total * nt) { p.ib = 0; p.lo = p.hi = p.t = S.n_tiles; p.pb = 0; return p; }
    long long rem = pos;
    p.lo = 0; p.hi = f0_first_block_end(S);
    while (rem >= S.total * (p.hi - p.lo) && p.hi < S.n_tiles) { rem -= S.total * (p.hi - p.lo); p.lo = p.hi; p.hi = min(S.n_tiles, p.hi + S.gb); }
    const long long len = p.hi - p.lo;
    const long long row = S.total / S.n_pb * len;                       // one template block of every bd
    p.pb = (int)min(rem / row, (long long)S.n_pb - 1);
    rem -= p.pb * row;
    int lo = 0, hi = S.n_bds - 1;                                       // bds[i].cum / n_pb = sum of w over the earlier entries
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (S.bds[mid].cum / S.n_pb * len <= rem) lo = mid; else hi = mid - 1; }
    rem -= S.bds[lo].cum / S.n_pb * len;
    p.ib = lo;
    p.t = p.lo + (int)min(rem / S.bds[lo].w, len - 1);
    f0_granule_up(S, p);
    return p;
  }
  if (pos >= S.total * nt) { p.ib = S.n_bds; p.lo = 0; p.hi = f0_first_block_end(S); p.pb = 0; p.t = 0; return p; }
  int lo = 0, hi = S.n_bds - 1;
  while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (S.bds[mid].cum * nt <= pos) lo = mid; else hi = mid - 1; }
  const SchedBd B = S.bds[lo];
  long long rem = pos - B.cum * nt;
  const long long cw = (long long)B.n_pb * B.w;
  p.ib = lo; p.lo = 0; p.hi = f0_first_block_end(S);
  while (rem >= cw * (p.hi - p.lo) && p.hi < S.n_tiles) { rem -= cw * (p.hi - p.lo); p.lo = p.hi; p.hi = min(S.n_tiles, p.hi + S.gb); }
  const int len = p.hi - p.lo;
  p.pb = min((int)(rem / ((long long)B.w * len)), B.n_pb - 1);
  p.t = p.lo + min((int)((rem - (long long)p.pb * B.w * len) / B.w), len - 1);
  f0_granule_up(S, p);
  return p;
}

// iterates this cluster's segments: (bd entry, template block, tiles [t0, t1))
struct F0Iter {
  F0Pos cur, end;
  bool pb_major;                            // F0Sched::n_pb > 0: cells are ordered (lo, pb, ib), else (ib, lo, pb)
  __device__ __forceinline__ bool at_end() const
  {
    if (pb_major)
      return cur.lo > end.lo || (cur.lo == end.lo && (cur.pb > end.pb || (cur.pb == end.pb && (cur.ib > end.ib || (cur.ib == end.ib && cur.t >= end.t)))));
    return cur.ib > end.ib || (cur.ib == end.ib && (cur.lo > end.lo || (cur.lo == end.lo && (cur.pb > end.pb || (cur.pb == end.pb && cur.t >= end.t)))));
  }
  __device__ __forceinline__ int seg_end() const { return (cur.ib == end.ib && cur.lo == end.lo && cur.pb == end.pb) ? end.t : cur.hi; }
};
#define FOR_F0_SEGMENTS(it, S, A, B)                                                              \
  for (F0Iter it{A, B, (S).n_pb > 0}; !it.at_end(); f0_next_cell(S, it.cur))                                    \
    if (it.cur.t >= it.seg_end()) continue; else

// ---- low-rate kernel schedule: per rate class the f0 kernel's order ((bin, detector), time block, template block, tile) ------
// A class is a low rate: its cells are (group = the same-rate slices of a (bin, detector), template block), all with the
// class's tile count.  The flattened sequence is class after class; cluster i takes the cost range [T i / G, T (i + 1) / G).
// Inside a class the time block is one cluster's share of tiles, so the clusters that reconstruct the template blocks of a
// group run side by side on the same y tiles (one reads a tile from DRAM, the others from L2) -- before, the units
// (group, template block) followed one another whole, the 8 template blocks of a group were at different tiles at any
// moment and y came from DRAM about 4.5 times (config 2: 267 MB of reads per launch for 75 MB of operands).
struct LowSched {
  const SchedBd* cells;                     // per class: one entry per group {first unit, template blocks, cost per tile, cum}
  int n_cls;
  int cell_begin[kNLowRates + 1];
  int n_tiles[kNLowRates], gb[kNLowRates];
  long long total[kNLowRates];              // sum of n_pb * w over the class's groups
  long long base[kNLowRates + 1];           // cost before class c (total * n_tiles summed); base[n_cls] = T
};

struct LowIter {                            // yields this cluster's segments (unit, tiles [t0, t1)) in schedule order
  const LowSched& L;
  long long PA, PB;
  int c;
  F0Sched S;
  F0Iter it;
  bool open;
  __device__ __forceinline__ LowIter(const LowSched& l, long long pa, long long pb) : L(l), PA(pa), PB(pb), c(-1), S{}, it{}, open(false) {}
  __device__ __forceinline__ bool open_next_class()
  {
    while (++c < L.n_cls) {
      const long long lo = max(PA, L.base[c]) - L.base[c], hi = min(PB, L.base[c + 1]) - L.base[c];
      if (lo >= hi) continue;
      S.bds = L.cells + L.cell_begin[c]; S.n_bds = L.cell_begin[c + 1] - L.cell_begin[c];
      S.n_tiles = L.n_tiles[c]; S.gb = L.gb[c]; S.gt = 1; S.n_pb = 0; S.total = L.total[c]; S.a0 = 0;
      it.cur = f0_locate(S, lo); it.end = f0_locate(S, hi); it.pb_major = false;
      return true;
    }
    return false;
  }
  __device__ __forceinline__ bool next(int& u, int& t0, int& t1)
  {
    for (;;) {
      if (!open) { if (!open_next_class()) return false; open = true; }
      else f0_next_cell(S, it.cur);
      while (!it.at_end() && it.cur.t >= it.seg_end()) f0_next_cell(S, it.cur);
      if (it.at_end()) { open = false; continue; }
      u = S.bds[it.cur.ib].bd + it.cur.pb; t0 = it.cur.t; t1 = it.seg_end();
      return true;
    }
  }
};
#define FOR_LOW_SEGMENTS(u, t0, t1)                                                               \
  for (LowIter li_(a.sched, PA, PB); ;)                                                           \
    if (int u = 0, t0 = 0, t1 = 0; !li_.next(u, t0, t1)) break; else

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
  uint64_t acc_full[PK_NACC_MAX], acc_empty[PK_NACC_MAX], ybar[PK_NACC_MAX];
  uint64_t consts, unit_done, r_ready;
  uint32_t py_tiles, pad_;                  // tiles the PY thread has started (read by the L2 prefetcher)
};

// Barrier counts: a "full" barrier of the leader gets its own producers' arrive.expect_tx plus the peer's relay, the peer's
// own copy only its producers'.  acc_empty lives in the leader: one arrival per epilogue warp of both CTAs.  unit_done is
// committed by the thread that finishes the unit's LAST tile, after it has seen the other thread's last tile complete.
__device__ __forceinline__ void pair_setup(PairBars& B, uint32_t* tmem_slot, int nsy, uint32_t rank, int warp, int tid, uint32_t n_pq, uint32_t n_drain)
{
  if (warp == 0) tmem_alloc2(tmem_slot, 512);
  if (tid == 32) {
    B.py_tiles = 0u;
    const uint32_t relay = rank == 0 ? 1u : 0u;
    for (int s = 0; s < nsy; ++s) { mbar_init(smem_u32(&B.yfull[s]), 1u + relay); mbar_init(smem_u32(&B.yempty[s]), 1); }
    for (int s = 0; s < PK_NQB; ++s) { mbar_init(smem_u32(&B.qfull[s]), n_pq + relay); mbar_init(smem_u32(&B.qempty[s]), 1); }
    for (int b = 0; b < PK_NACC_MAX; ++b) {
      mbar_init(smem_u32(&B.acc_full[b]), 1); mbar_init(smem_u32(&B.acc_empty[b]), n_drain); mbar_init(smem_u32(&B.ybar[b]), 1);
    }
    mbar_init(smem_u32(&B.consts), 1u + relay);
    mbar_init(smem_u32(&B.unit_done), 1);
    mbar_init(smem_u32(&B.r_ready), 16);          // RT: "the unit's R is in TMEM": one arrival per epilogue warp of both CTAs
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

// y stages of a slice with nm = L_pad / 16 MMAs per tile: ceil(nm / 8) stages of nearly equal size (<= 8 MMAs, K <= 128)
__host__ __device__ inline int stage_count(int nm, int cap) { return (nm + cap - 1) / cap; }

// m back-to-back MMAs of one y stage: D (+)= R[l-groups from a_lo] * stage^T, N = 128.  a_lo: descriptor of R at this K
// offset (LBO 2048: 128 rows per l-group, 256 sixteen-byte units per K = 16); b_lo: the stage (LBO 1024: 64 rows, 128 units)
// RT: a_lo is the TMEM address of R's columns for this K offset (8 columns per K = 16).
template <bool RT>
__device__ __forceinline__ void mma_y_stage(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, int m, uint32_t acc0)
{
  if constexpr (RT) mma2_ts(d_tmem, a_lo, desc64(b_lo), idesc, acc0); else mma2_ss(d_tmem, desc64(a_lo), desc64(b_lo), idesc, acc0);
#pragma unroll 4
  for (int k = 1; k < m; ++k) {
    a_lo += RT ? 8u : 256u; b_lo += 128u;
    if constexpr (RT) mma2_ts(d_tmem, a_lo, desc64(b_lo), idesc, 1u); else mma2_ss(d_tmem, desc64(a_lo), desc64(b_lo), idesc, 1u);
  }
}

// ------------------------------------------------------------------------------------------------
struct SegSrc {                             // per-role copy of the current unit's operand sources (this CTA's halves)
  const uint8_t* Y0;                        // Y16 record of the unit's rate group: 64-row tile 0 (lloid_api.cu: the slices' y lie side by side)
  const uint8_t* Rsrc[kMaxGroupSlices];     // this CTA's 128-row block of the slice's R16
  int nm[kMaxGroupSlices];                  // L_pad / 16
  int n, stages_per_tile;
  uint32_t rbytes, ystep;                   // bytes of the unit's R block; bytes from one 64-row y tile to the next
  uint64_t mlist;                           // MMAs per stage minus one, 4 bits per stage, in the order of the tile's stages (<= 16)
};

// The K = sum L_pad of a unit is one contiguous operand (y record in HBM, R in shared memory / TMEM), cut into
// ceil(nm / ycap) stages of nearly equal size whatever the slice boundaries.
__device__ __forceinline__ void seg_fill(SegSrc& S, const SliceParams* __restrict__ sp, const int32_t* slice, int n, int rb, int ycap)
{
  S.n = n; S.rbytes = 0; S.mlist = 0;
  int nm_all = 0;
  for (int i = 0; i < n; ++i) {             // one thread
    const SliceParams* P = sp + slice[i];
    const int L = P->L_pad;
    if (i == 0) { S.Y0 = reinterpret_cast<const uint8_t*>(P->Y); S.ystep = (uint32_t)P->y_step64; }
    S.Rsrc[i] = reinterpret_cast<const uint8_t*>(P->R16) + (size_t)rb * L * 256;
    S.nm[i] = L >> 4;
    nm_all += L >> 4;
    S.rbytes += (uint32_t)L * 256u;
  }
  const int nst = stage_count(nm_all, ycap), base = nm_all / nst, ext = nm_all - base * nst;
  for (int j = 0; j < nst; ++j) S.mlist |= (uint64_t)(base + (j < ext ? 1 : 0) - 1) << (4 * j);
  S.stages_per_tile = nst;
}

struct YAddr { uint32_t full0, empty0, dst0, step; };   // barrier arrays and slots of the y ring (dst: address, or descriptor for IY)

// PY role of both kernels: y stages of the unit's slices for tiles [t0, t1) (this CTA's 64-row half of every 128-row
// tile), and the stationary R of the unit.  R goes out after `pre` stages of the new unit are in flight: the ring refills
// while the previous unit drains.  extra/extra_bytes: loaded once with the first R (the f0 kernel's band matrices).
// RT (R in TMEM, loaded by the epilogue warps): only the band matrices go out, with the first unit.
template <bool RT>
__device__ __forceinline__ void py_segment(YRing& rg, const YAddr ya, int& seg_i, const SegSrc& sg, uint32_t consts_u, uint32_t unit_done_u, uint32_t sR_u, uint32_t progress_u,
                                           uint32_t rank, int t0, int t1, uint32_t extra_dst, const uint8_t* extra, uint32_t extra_bytes,
                                           bool trace, long long* tw)
{
  int pre = (seg_i == 0) ? 0 : min((int)rg.n, sg.stages_per_tile);
  bool need_R = true;
  if constexpr (RT) {
    need_R = false;
    if (seg_i == 0) {
      if (extra_bytes) { mbar_expect_tx(consts_u, extra_bytes); copy_pieces(extra_dst, extra, extra_bytes, consts_u); }
      else mbar_arrive(consts_u);
    }
  }
  auto load_R = [&]() {
    if (seg_i > 0) TWAIT(1, unit_done_u, (uint32_t)(seg_i - 1) & 1u);   // every MMA that reads the old R is complete
    const int n_r = sg.n;
    mbar_expect_tx(consts_u, sg.rbytes + (seg_i == 0 ? extra_bytes : 0u));
    uint32_t off = 0;
    for (int i = 0; i < n_r; ++i) {
      copy_pieces(sR_u + off, sg.Rsrc[i], (uint32_t)sg.nm[i] * 4096u, consts_u);
      off += (uint32_t)sg.nm[i] * 4096u;
    }
    if (seg_i == 0 && extra_bytes) copy_pieces(extra_dst, extra, extra_bytes, consts_u);
    need_R = false;
  };
  if (need_R && pre == 0) load_R();
  const uint32_t step2 = 2u * sg.ystep;
  const uint64_t mlist = sg.mlist;
  const int nst = sg.stages_per_tile;
  const uint8_t* src = sg.Y0 + (size_t)(2 * t0 + (int)rank) * sg.ystep;          // this CTA's 64-row half of tile t0
  for (int t = t0; t < t1; ++t, src += step2) {
    st_shared_u32(progress_u, ++rg.tiles);                 // paces the prefetcher (prefetch_segment)
    const uint8_t* p = src;
    uint64_t ml = mlist;
    for (int j = 0; j < nst; ++j, ml >>= 4) {
      const uint32_t bytes = ((uint32_t)(ml & 15u) + 1u) * 2048u;
      const uint32_t full = ya.full0 + 8u * rg.s;
      TWAIT(0, ya.empty0 + 8u * rg.s, rg.ph ^ 1u);
      { TSPAN_BEGIN(); mbar_expect_tx(full, bytes); TSPAN_END(3); }
      { TSPAN_BEGIN(); bulk_g2s(ya.dst0 + rg.s * ya.step, p, bytes, full); TSPAN_END(4); }
      rg.advance();
      p += bytes;
      if (need_R && --pre == 0) load_R();
    }
  }
  if (need_R) load_R();
  ++seg_i;
}

// relay role (peer CTA): forwards the completion of this CTA's y stages and R loads to the leader's barriers
template <bool RT>
__device__ __forceinline__ void relay_y_segment(YRing& rg, const YAddr ya, int& seg_i, int n_stages, uint32_t consts_u)
{
  // consts first (it is requested before or among the first stages of the unit and the leader needs it first); RT: once
  if (!RT || seg_i == 0) {
    mbar_wait(consts_u, (uint32_t)seg_i & 1u);
    mbar_arrive_cluster(consts_u & kLeaderMask);
  }
  for (int n = n_stages; n > 0; --n) {
    const uint32_t full = ya.full0 + 8u * rg.s;
    mbar_wait(full, rg.ph);
    mbar_arrive_cluster(full & kLeaderMask);
    rg.advance();
  }
  ++seg_i;
}

// L2 prefetcher (one thread of an otherwise idle warp, both CTAs): when PY starts tile t of a unit, the record of tile
// t + PK_YPF is requested from HBM.  (Issued by PY itself the instruction cost it ~580 cycles per tile in the low-rate
// kernel: cp.async.bulk.prefetch.L2 of a 20-40 KB record blocks the issuing thread.)  Paced by PY's progress word, which
// only grows: no barrier phase can be missed.
__device__ __forceinline__ void prefetch_segment(uint32_t& seen, uint32_t progress_u, const uint8_t* Y0, uint32_t ystep, uint32_t rank, int t0, int t1)
{
  const uint32_t step2 = 2u * ystep;
  const uint8_t* src = Y0 + (size_t)(2 * (t0 + PK_YPF) + (int)rank) * ystep;
  for (int t = t0; t < t1; ++t, src += step2) {
    ++seen;
    while (ld_shared_volatile_u32(progress_u) < seen) __nanosleep(64);
    if (t + PK_YPF < t1) bulk_prefetch_l2(src, ystep);
  }
}

// RT, epilogue warps at the start of a unit: the unit's R block of this CTA (128 rows x K) -> TMEM columns [PK_ACOL, PK_ACOL + K / 2).
// R16 is [l / 8][lane][8 fp16]: a thread (= lane) reads the 16 bytes of one l-group and stores them as four 32-bit columns;
// the two warp groups (wg) take alternate l-groups.  Called when every MMA of the previous unit is complete (the caller has
// just drained that unit's last accumulator); afterwards r_ready tells the issuing thread.
__device__ __forceinline__ void load_R_tmem(const SliceParams* __restrict__ sp, const int32_t* slice, int n, int rb,
                                            uint32_t tmem_lane_base, int lane_row, int wg)
{
  uint32_t col = tmem_lane_base + PK_ACOL;
  for (int i = 0; i < n; ++i) {
    const SliceParams* P = sp + slice[i];
    const int ng = P->L_pad >> 3;
    const uint4* __restrict__ src = reinterpret_cast<const uint4*>(reinterpret_cast<const uint8_t*>(P->R16) + (size_t)rb * P->L_pad * 256) + lane_row;
    int g = wg;
    for (; g + 6 < ng; g += 8) {             // four loads in flight
      const uint4 v0 = __ldg(src + (size_t)g * 128), v1 = __ldg(src + (size_t)(g + 2) * 128);
      const uint4 v2 = __ldg(src + (size_t)(g + 4) * 128), v3 = __ldg(src + (size_t)(g + 6) * 128);
      tmem_st4(col + 4u * g, v0.x, v0.y, v0.z, v0.w);
      tmem_st4(col + 4u * (g + 2), v1.x, v1.y, v1.z, v1.w);
      tmem_st4(col + 4u * (g + 4), v2.x, v2.y, v2.z, v2.w);
      tmem_st4(col + 4u * (g + 6), v3.x, v3.y, v3.z, v3.w);
    }
    for (; g < ng; g += 2) {
      const uint4 v = __ldg(src + (size_t)g * 128);
      tmem_st4(col + 4u * g, v.x, v.y, v.z, v.w);
    }
    col += 4u * ng;
  }
  tmem_st_wait();
}

// IY role: the y MMAs of one tile into accumulator d_tmem (first MMA overwrites).  mlist: the tile's stages in order, MMAs
// per stage minus one in 4 bits each (SegSrc::mlist, read once per unit: the loop touches no shared memory but the barriers)
template <bool RT>
__device__ __forceinline__ void iy_tile(YRing& rg, const YAddr ya, uint64_t mlist, int n_stages, uint32_t d_tmem, uint32_t a_base, uint32_t idesc,
                                        bool trace, long long* tw)
{
  uint32_t acc = 0u, a_lo = a_base;
  for (int j = 0; j < n_stages; ++j, mlist >>= 4) {
    const int m = (int)(mlist & 15u) + 1;
    TWAIT(2, ya.full0 + 8u * rg.s, rg.ph);
    fence_after();
#ifdef LLOID_TRACE_BUILD
    if (!(g_exp & 2))
#endif
    { TSPAN_BEGIN(); mma_y_stage<RT>(d_tmem, a_lo, ya.dst0 + rg.s * ya.step, idesc, m, acc); TSPAN_END(3); }
    { TSPAN_BEGIN(); commit2(ya.empty0 + 8u * rg.s, 3); TSPAN_END(4); }
    acc = 1u;
    a_lo += (uint32_t)m * (RT ? 8u : 256u);
    rg.advance();
  }
}

// ------------------------------------------------------------------------------------------------
struct LowPArgs {
  const SliceParams* sp; const RateGroup* groups; const LowUnit* units;
  int r_bytes, nsy, ystage, ycap, trace;
  LowSched sched;
};

template <bool RT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PK_THREADS, 1)
lowrate_pair_kernel(const __grid_constant__ LowPArgs a)
{
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) PairBars bars;
  __shared__ uint32_t tmem_slot;
  __shared__ SegSrc seg[3];                             // [0] PY, [1] IY, [2] relay

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = cluster_ctarank();
  const long long T_all = a.sched.base[a.sched.n_cls];
  const long long PA = T_all * (long long)(blockIdx.x >> 1) / (long long)(gridDim.x >> 1);
  const long long PB = T_all * (long long)((blockIdx.x >> 1) + 1) / (long long)(gridDim.x >> 1);
  if (PA >= PB) return;                                 // both CTAs of the cluster take the same decision

  const int nsy = a.nsy;
  pair_setup(bars, &tmem_slot, nsy, rank, warp, tid, 1u, 16u);          // all 8 epilogue warps of both CTAs drain every tile
  const uint32_t tmem = tmem_slot;
  constexpr uint32_t NACC = Acc<RT>::N;
  const uint32_t sR_u = smem_u32(smem);                 // !RT: [l_sum / 8][128 rows][8] fp16
  const uint32_t ring_u = sR_u + (RT ? 0u : (uint32_t)a.r_bytes);
  const uint32_t consts_u = smem_u32(&bars.consts), unit_done_u = smem_u32(&bars.unit_done), r_ready_u = smem_u32(&bars.r_ready);
  const uint32_t progress_u = smem_u32(&bars.py_tiles);
  const YAddr ya{smem_u32(&bars.yfull[0]), smem_u32(&bars.yempty[0]), ring_u, (uint32_t)a.ystage};

  if (warp == 0) {
    if (elect_one()) {
      YRing rg{0u, 0u, (uint32_t)nsy};
      int seg_i = 0, nt = 0;
      TRACE_BEGIN();
      FOR_LOW_SEGMENTS(u, t0, t1) {
        const LowUnit un = a.units[u];
        const RateGroup* G = a.groups + un.group;
        seg_fill(seg[0], a.sp, G->slice, G->n_slices, 2 * un.pb + (int)rank, a.ycap);
        py_segment<RT>(rg, ya, seg_i, seg[0], consts_u, unit_done_u, sR_u, progress_u, rank, t0, t1, 0u, nullptr, 0u, trace, tw);
        nt += t1 - t0;
      }
      if (rank == 0) TRACE_END(0, 0, nt);
    }
  } else if (warp == 7) {
    if (elect_one()) {
      uint32_t seen = 0;
      FOR_LOW_SEGMENTS(u, t0, t1) {
        const SliceParams* P = a.sp + a.groups[a.units[u].group].slice[0];
        prefetch_segment(seen, progress_u, reinterpret_cast<const uint8_t*>(P->Y), (uint32_t)P->y_step64, rank, t0, t1);
      }
    }
  } else if (warp == 4 && rank == 1) {
    if (elect_one()) {
      YRing rg{0u, 0u, (uint32_t)nsy};
      int seg_i = 0;
      FOR_LOW_SEGMENTS(u, t0, t1) {
        const LowUnit un = a.units[u];
        const RateGroup* G = a.groups + un.group;
        seg_fill(seg[2], a.sp, G->slice, G->n_slices, 2 * un.pb + (int)rank, a.ycap);
        relay_y_segment<RT>(rg, ya, seg_i, (t1 - t0) * seg[2].stages_per_tile, consts_u);
      }
    }
  } else if (warp == 1 && rank == 0) {
    // ===== IY: the MMAs (one elected thread of the leader CTA).  A second issuing thread for the odd tiles was 10 % faster
    // but faulted (cudaErrorLaunchFailure) once in a few hundred launches on the full config-2 bank; not understood. =====
    if (elect_one()) {
      SegSrc& sg = seg[1];
      const uint32_t idesc = idesc_f16_pair(128);
      const uint32_t a_base = RT ? tmem + PK_ACOL : desc_lo(sR_u, 2048u);
      const uint32_t acc_full_u = smem_u32(&bars.acc_full[0]), acc_empty_u = smem_u32(&bars.acc_empty[0]);
      const YAddr yd{ya.full0, ya.empty0, desc_lo(ring_u, 1024u), (uint32_t)a.ystage >> 4};   // dst = descriptor of the stage
      YRing rg{0u, 0u, (uint32_t)nsy};
      int seg_i = 0;
      uint32_t e = 0;
      TRACE_BEGIN();
      FOR_LOW_SEGMENTS(u, t0, t1) {
        const LowUnit un = a.units[u];
        const RateGroup* G = a.groups + un.group;
        seg_fill(sg, a.sp, G->slice, G->n_slices, 2 * un.pb, a.ycap);
        const uint64_t mlist = sg.mlist;
        const int n_stages = sg.stages_per_tile;
        if constexpr (RT) TWAIT(0, r_ready_u, (uint32_t)seg_i & 1u); else TWAIT(0, consts_u, (uint32_t)seg_i & 1u);   // the unit's R is in place
        fence_after();
        for (int t = t0; t < t1; ++t, ++e) {
          const uint32_t b = e & (NACC - 1), ph = (e / NACC) & 1u;
          TWAIT(1, acc_empty_u + 8u * b, ph ^ 1u);
          fence_after();
          iy_tile<RT>(rg, yd, mlist, n_stages, tmem + b * 128u, a_base, idesc, trace, tw);
          commit2(acc_full_u + 8u * b, 3);
        }
        if constexpr (!RT) commit2(unit_done_u, 3);
        ++seg_i;
      }
      TRACE_END(0, 1, (int)e);
    }
  } else if (warp >= 8 && warp < 16) {
    // ===== epilogue: thread = row; warps 8-11 columns [0, 64), warps 12-15 columns [64, 128); fp32 -> fp16 -> Q16 =====
    const int q = warp & 3, wg = (warp - 8) >> 2;
    const int row = q * 32 + lane;
    const uint32_t acc_empty_leader = smem_u32(&bars.acc_empty[0]) & kLeaderMask;
    const uint32_t acc_full_u = smem_u32(&bars.acc_full[0]);
    uint32_t e = 0;
    TRACE_BEGIN();
    FOR_LOW_SEGMENTS(u, t0, t1) {
      const LowUnit un = a.units[u];
      const RateGroup* Gp = a.groups + un.group;
      const int q_cap = Gp->q_groups_cap;
      if constexpr (RT) {
        // this warp has drained the previous unit's last accumulator, so every MMA that read the old R is complete
        __syncwarp();
        load_R_tmem(a.sp, Gp->slice, Gp->n_slices, 2 * un.pb + (int)rank, tmem + ((uint32_t)(q * 32) << 16), row, wg);
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(r_ready_u & kLeaderMask);
      }
      __half* __restrict__ Q = Gp->Q + ((size_t)(2 * un.pb + (int)rank) * q_cap * 128 + row) * 8;
      for (int t = t0; t < t1; ++t, ++e) {
        const uint32_t b = e & (NACC - 1), ph = (e / NACC) & 1u;
        TWAIT(0, acc_full_u + 8u * b, ph);
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
    if (rank == 0 && tid == 256) TRACE_END(0, 4, (int)e);
  }
  pair_teardown(tmem, warp);
}

constexpr int kIqFast = 3;                  // interpolation MMAs per rate and tile held in registers (d >= 4: at most 3 chunks)

// ------------------------------------------------------------------------------------------------
struct F0PArgs {
  const SliceParams* sp; const BdPlan* bd; const RateGroup* groups;
  const uint8_t* P;                                     // [2][p_bytes]: band-matrix blob of rank 0, of rank 1
  Peak* partials; Capture cap; long long k_a;
  int n_lr, c, r_bytes, p_bytes, q_bytes, nsy, ystage, ycap, slots_cap, max_templates, trace;
  uint32_t q_gate;                                      // bits of theta^2 (1 - 2^-16): |rho|^2 at or below it cannot trigger
  F0Sched sched;
  PairRate rate[kNLowRates];
  PairMma tab[kPairTabMax];                             // interpolation MMAs, see PairMma
};

template <bool CAPTURE, bool RT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PK_THREADS, 1)
f0_pair_kernel(const __grid_constant__ F0PArgs a)
{
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ __align__(8) PairBars bars;
  __shared__ uint32_t tmem_slot;
  __shared__ SegSrc seg[3];                             // [0] PY, [1] IY, [2] relay
  __shared__ F0Pos s_pos[2];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = cluster_ctarank();
  const F0Sched& S = a.sched;
  const long long a0 = S.a0;
  if (tid == 0) {
    const long long T = S.total * S.n_tiles;
    const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;
    s_pos[0] = f0_locate(S, T * (long long)cid / ncl);
    s_pos[1] = f0_locate(S, T * (long long)(cid + 1) / ncl);
  }
  __syncthreads();
  const F0Pos pA = s_pos[0], pB = s_pos[1];
  { F0Iter it{pA, pB, S.n_pb > 0}; if (it.at_end()) return; }       // both CTAs of the cluster take the same decision

  const int nsy = a.nsy, n_lr = a.n_lr, gt = S.gt;
  constexpr uint32_t NACC = Acc<RT>::N;
  const uint32_t sR_u = smem_u32(smem);                 // !RT: [l_sum / 8][128 rows][8] fp16
  const uint32_t sP_u = sR_u + (RT ? 0u : (uint32_t)a.r_bytes);     // this rank's band-matrix blocks
  const uint32_t sQ_u = sP_u + (uint32_t)a.p_bytes;     // per-rate circular buffers of 16-row chunks (4 KB each)
  const uint32_t ring_u = sQ_u + (uint32_t)a.q_bytes;   // y ring
  pair_setup(bars, &tmem_slot, nsy, rank, warp, tid, 2u, 8u);           // 4 epilogue warps of each CTA drain a tile (the two groups alternate)
  const uint32_t tmem = tmem_slot;
  const uint32_t consts_u = smem_u32(&bars.consts), unit_done_u = smem_u32(&bars.unit_done), r_ready_u = smem_u32(&bars.r_ready);
  const uint32_t progress_u = smem_u32(&bars.py_tiles);
  const YAddr ya{smem_u32(&bars.yfull[0]), smem_u32(&bars.yempty[0]), ring_u, (uint32_t)a.ystage};
  const uint32_t qfull_u = smem_u32(&bars.qfull[0]), qempty_u = smem_u32(&bars.qempty[0]);
  const uint32_t acc_full_u = smem_u32(&bars.acc_full[0]), ybar_u = smem_u32(&bars.ybar[0]);

  if (warp == 0) {
    // ===== PY: y tiles of the d = 1 slices, R and P =====
    if (elect_one()) {
      YRing rg{0u, 0u, (uint32_t)nsy};
      int seg_i = 0, nt = 0;
      TRACE_BEGIN();
      FOR_F0_SEGMENTS(it, S, pA, pB) {
        const int t0 = it.cur.t, t1 = it.seg_end(), bdi = S.bds[it.cur.ib].bd;
        const BdPlan* B = a.bd + bdi;
        seg_fill(seg[0], a.sp, B->f0_slice, B->n_f0, 2 * it.cur.pb + (int)rank, a.ycap);
        py_segment<RT>(rg, ya, seg_i, seg[0], consts_u, unit_done_u, sR_u, progress_u, rank, t0, t1, sP_u, a.P + (size_t)rank * a.p_bytes, (uint32_t)a.p_bytes, trace, tw);
        nt += t1 - t0;
      }
      if (rank == 0) TRACE_END(1, 0, nt);
    }
  } else if (warp == 7) {
    if (elect_one()) {
      uint32_t seen = 0;
      FOR_F0_SEGMENTS(it, S, pA, pB) {
        const SliceParams* P = a.sp + a.bd[S.bds[it.cur.ib].bd].f0_slice[0];
        prefetch_segment(seen, progress_u, reinterpret_cast<const uint8_t*>(P->Y), (uint32_t)P->y_step64, rank, it.cur.t, it.seg_end());
      }
    }
  } else if (warp == 4 && rank == 1) {
    if (elect_one()) {
      YRing rg{0u, 0u, (uint32_t)nsy};
      int seg_i = 0;
      FOR_F0_SEGMENTS(it, S, pA, pB) {
        const int t0 = it.cur.t, t1 = it.seg_end(), bdi = S.bds[it.cur.ib].bd;
        const BdPlan* B = a.bd + bdi;
        seg_fill(seg[2], a.sp, B->f0_slice, B->n_f0, 2 * it.cur.pb + (int)rank, a.ycap);
        relay_y_segment<RT>(rg, ya, seg_i, (t1 - t0) * seg[2].stages_per_tile, consts_u);
      }
    }
  } else if (warp == 2 || warp == 6) {
    // ===== PQ0 / PQ1 (even / odd rates): the rows of a rate's rho^(d) window that tile e needs and tile e - 1 did not have =====
    if (elect_one()) {
      const int rsel = warp == 2 ? 0 : 1;
      uint32_t e = 0;
      TRACE_BEGIN();
      int adv[kNLowRates], cap[kNLowRates], cnext[kNLowRates], slot[kNLowRates];
      uint32_t base[kNLowRates];
#pragma unroll
      for (int r = 0; r < kNLowRates; ++r) { adv[r] = a.rate[r].adv; cap[r] = a.rate[r].cap_chunks; base[r] = sQ_u + (uint32_t)a.rate[r].ring_off; cnext[r] = 0; slot[r] = 0; }
      FOR_F0_SEGMENTS(it, S, pA, pB) {
        const int t0 = it.cur.t, t1 = it.seg_end(), bdi = S.bds[it.cur.ib].bd, rb = 2 * it.cur.pb + (int)rank;
        const uint8_t* qsrc[kNLowRates];
#pragma unroll
        for (int r = 0; r < kNLowRates; ++r) {
          qsrc[r] = nullptr;
          if (r < n_lr && (r & 1) == rsel) {
            const RateGroup* G = a.groups + bdi * n_lr + r;
            if (G->n_slices > 0) qsrc[r] = reinterpret_cast<const uint8_t*>(G->Q) + (size_t)rb * G->q_groups_cap * 2048;
            cnext[r] = (adv[r] * t0) >> 4;              // the unit's first tile fetches its whole window
            slot[r] = cnext[r] % cap[r];
          }
        }
        for (int t = t0; t < t1; ++t, ++e) {
          // a unit's first tile fetches whole windows into slots earlier tiles may still be reading: drain first.  (The
          // even and the odd tiles finish on different threads: both of the last two must be complete.)
          if (t == t0) {
            if (e > 1) TWAIT(1, qempty_u + 8u * ((e - 2) & (PK_NQB - 1)), ((e - 2) >> 2) & 1u);
            if (e > 0) TWAIT(1, qempty_u + 8u * ((e - 1) & (PK_NQB - 1)), ((e - 1) >> 2) & 1u);
          } else {
            // tile e's rows overwrite chunks that only tiles <= e - PK_QDIST read.  Even and odd tiles are finished by different
            // threads, each in order: BOTH of e - PK_QDIST and e - PK_QDIST - 1 must be complete.  (Waiting for the first one
            // only let a lagging thread's tile lose rows of its window while its MMAs were still to run: about one wrong SNR
            // value in 10^8, seen as triggers that came and went between identical runs.)
            if (e >= PK_QDIST + 1) TWAIT(0, qempty_u + 8u * ((e - PK_QDIST - 1) & (PK_NQB - 1)), ((e - PK_QDIST - 1) >> 2) & 1u);
            if (e >= PK_QDIST) TWAIT(0, qempty_u + 8u * ((e - PK_QDIST) & (PK_NQB - 1)), ((e - PK_QDIST) >> 2) & 1u);
          }
          const uint32_t fb = qfull_u + 8u * (e & (PK_NQB - 1));
          int nnew[kNLowRates];
          uint32_t total = 0;
#pragma unroll
          for (int r = 0; r < kNLowRates; ++r) {
            nnew[r] = qsrc[r] ? ((adv[r] * (t + 1) + 31) >> 4) - cnext[r] : 0;
            total += (uint32_t)nnew[r];
          }
          if (((t - t0) & 3) == 0) {
            // pull the rows tiles t + PK_QPF .. + 3 will ask for from HBM into L2 now: the shared-memory windows only
            // hold PK_QDIST tiles of lookahead, far less than the DRAM latency under load
#pragma unroll
            for (int r = 0; r < kNLowRates; ++r) {
              if (!qsrc[r]) continue;
              const int tf = min(t + PK_QPF, t1), tg = min(t + PK_QPF + 4, t1);
              const int c0 = (adv[r] * tf + 31) >> 4, c1 = (adv[r] * tg + 31) >> 4;             // chunks_upto(tf - 1), chunks_upto(tg - 1)
              if (c1 > c0) bulk_prefetch_l2(qsrc[r] + (size_t)c0 * 4096, (uint32_t)(c1 - c0) * 4096u);
            }
          }
          mbar_expect_tx(fb, total * 4096u);            // total == 0: a plain arrival
#pragma unroll
          for (int r = 0; r < kNLowRates; ++r) {
            if (nnew[r] <= 0) continue;
            const uint8_t* src = qsrc[r] + (size_t)cnext[r] * 4096;
            const int n1 = min(nnew[r], cap[r] - slot[r]);
            bulk_g2s(base[r] + (uint32_t)slot[r] * 4096u, src, (uint32_t)n1 * 4096u, fb);
            if (nnew[r] > n1) bulk_g2s(base[r], src + (size_t)n1 * 4096, (uint32_t)(nnew[r] - n1) * 4096u, fb);
            cnext[r] += nnew[r];
            slot[r] += nnew[r]; if (slot[r] >= cap[r]) slot[r] -= cap[r];
          }
        }
      }
      if (rank == 0 && rsel == 0) TRACE_END(1, 2, (int)e);
    }
  } else if (warp == 5 && rank == 1) {
    // ===== relay of the rho^(d) tile events =====
    if (elect_one()) {
      uint32_t e = 0;
      FOR_F0_SEGMENTS(it, S, pA, pB) {
        for (int t = it.cur.t; t < it.seg_end(); ++t, ++e) {
          const uint32_t fb = qfull_u + 8u * (e & (PK_NQB - 1));
          mbar_wait(fb, (e >> 2) & 1u);
          mbar_arrive_cluster(fb & kLeaderMask);
        }
      }
    }
  } else if (warp == 1 && rank == 0) {
    // ===== IY: MMAs of the d = 1 slices.  ONE thread here: this role spends most of its time blocked on the pipe (N = 128
    // MMAs with both operands in shared memory take all of its 128 B/clk: 4 KB of A, 2 KB of B for this SM and 2 KB for
    // the peer per 64 cycles), and with a second issuing thread for the odd tiles the f0 kernel faulted on the full
    // config-2 bank (cudaErrorLaunchFailure, not understood; the low-rate kernel runs two) =====
    if (elect_one()) {
      SegSrc& sg = seg[1];
      const uint32_t idesc = idesc_f16_pair(128);
      const uint32_t a_base = RT ? tmem + PK_ACOL : desc_lo(sR_u, 2048u);
      const uint32_t acc_empty_u = smem_u32(&bars.acc_empty[0]);
      const YAddr yd{ya.full0, ya.empty0, desc_lo(ring_u, 1024u), (uint32_t)a.ystage >> 4};
      YRing rg{0u, 0u, (uint32_t)nsy};
      int seg_i = 0;
      uint32_t e = 0;
      TRACE_BEGIN();
      FOR_F0_SEGMENTS(it, S, pA, pB) {
        const int t0 = it.cur.t, t1 = it.seg_end(), bdi = S.bds[it.cur.ib].bd;
        const BdPlan* B = a.bd + bdi;
        seg_fill(sg, a.sp, B->f0_slice, B->n_f0, 2 * it.cur.pb, a.ycap);
        const uint64_t mlist = sg.mlist;
        const int n_stages = sg.stages_per_tile;
        if constexpr (RT) TWAIT(0, r_ready_u, (uint32_t)seg_i & 1u); else TWAIT(0, consts_u, (uint32_t)seg_i & 1u);   // the unit's R is in place
        fence_after();
        for (int t = t0; t < t1; ++t, ++e) {
          const uint32_t b = e & (NACC - 1), ph = (e / NACC) & 1u;
          TWAIT(1, acc_empty_u + 8u * b, ph ^ 1u);
          fence_after();
          iy_tile<RT>(rg, yd, mlist, n_stages, tmem + b * 128u, a_base, idesc, trace, tw);
          commit2(ybar_u + 8u * b, 1);
        }
        ++seg_i;
      }
      TRACE_END(1, 1, (int)e);
    }
  } else if ((warp == 3 || warp == 5) && rank == 0) {
    // ===== IQ0 / IQ1: interpolation MMAs (A4) of the even / odd tiles, after the tile's y part is complete.  (Two threads
    // accumulating into the SAME accumulator concurrently gave wrong sums: the pipe orders the MMAs of one thread only;
    // tiles of different parity use different accumulators.) =====
    if (elect_one()) {
      const uint32_t which = warp == 3 ? 0u : 1u;
      uint32_t e = 0;
      int adv[kNLowRates], cap[kNLowRates], sb[kNLowRates], vmask[kNLowRates], mine_n = 0;
      uint32_t qa[kNLowRates];
#pragma unroll
      for (int r = 0; r < kNLowRates; ++r) {
        adv[r] = a.rate[r].adv; cap[r] = a.rate[r].cap_chunks; vmask[r] = a.rate[r].n_var - 1; sb[r] = 0;
        qa[r] = desc_lo(sQ_u + (uint32_t)a.rate[r].ring_off, 2048u);
      }
      const uint32_t p_base = sP_u >> 4;
      TRACE_BEGIN();
      if constexpr (RT) { mbar_wait(consts_u, 0u); fence_after(); }   // the band matrices of both CTAs have landed (!RT: they come with the first R)
      FOR_F0_SEGMENTS(it, S, pA, pB) {
        const int t0 = it.cur.t, t1 = it.seg_end(), bdi = S.bds[it.cur.ib].bd;
        uint32_t mine = 0;
#pragma unroll
        for (int r = 0; r < kNLowRates; ++r)
          if (r < n_lr && a.groups[bdi * n_lr + r].n_slices > 0) { mine |= 1u << r; sb[r] = ((adv[r] * t0) >> 4) % cap[r]; }
        for (int t = t0; t < t1; ++t, ++e) {
          if ((e & 1u) == which) {
            const uint32_t b = e & (NACC - 1), ph = (e / NACC) & 1u;
            const uint32_t d_tmem = tmem + b * 128u;
            // the tile's interpolation MMAs, read from the table BEFORE the waits: the indexed constant loads (a dependent
            // chain of ~2000 cycles per tile when they sat between the wait and the MMAs) overlap the wait for the y part
            PairMma im[kNLowRates][kIqFast];
            int nit[kNLowRates], ix[kNLowRates];
#pragma unroll
            for (int r = 0; r < kNLowRates; ++r) {
              nit[r] = 0; ix[r] = 0;
              if (!(mine >> r & 1u)) continue;
              const int v = t & vmask[r];
              nit[r] = a.rate[r].n_items[v];
              ix[r] = a.rate[r].tab_off[v] + sb[r] * nit[r];                 // [slot of the window's first chunk][item]
#pragma unroll
              for (int k = 0; k < kIqFast; ++k) if (k < nit[r]) im[r][k] = a.tab[ix[r] + k];
            }
            TWAIT(0, ybar_u + 8u * b, ph);
            fence_after();
            // the tile's window holds rows that arrived with THIS tile's event and with the previous tile's, which the other
            // IQ thread waited for, not this one -- and bulk copies complete in any order: wait for both.  (With the wait for
            // the own event only, a window row could still be in flight when its MMA ran: see the note in the PQ role.)
            if (e > 0) TWAIT(1, qfull_u + 8u * ((e - 1) & (PK_NQB - 1)), ((e - 1) >> 2) & 1u);
            TWAIT(1, qfull_u + 8u * (e & (PK_NQB - 1)), (e >> 2) & 1u);
            fence_after();
            {
              TSPAN_BEGIN();
#ifdef LLOID_TRACE_BUILD
              if (!(g_exp & 1))
#endif
#pragma unroll
              for (int r = 0; r < kNLowRates; ++r) {
#pragma unroll
                for (int k = 0; k < kIqFast; ++k)
                  if (k < nit[r]) mma2_ss(d_tmem + im[r][k].d_col, desc64(qa[r] + im[r][k].a_off), desc64(p_base + im[r][k].p_lo), im[r][k].idesc, 1u);
                for (int k = kIqFast; k < nit[r]; ++k) {                     // d = 2 windows (5 chunks), when that rate is not folded
                  const PairMma m = a.tab[ix[r] + k];
                  mma2_ss(d_tmem + m.d_col, desc64(qa[r] + m.a_off), desc64(p_base + m.p_lo), m.idesc, 1u);
                }
              }
              TSPAN_END(2);
            }
            { TSPAN_BEGIN(); commit2(qempty_u + 8u * (e & (PK_NQB - 1)), 3); commit2(acc_full_u + 8u * b, 3); TSPAN_END(3); }
            ++mine_n;
          }
          // window start of the next tile: floor(adv (t + 1) / 16) chunks
#pragma unroll
          for (int r = 0; r < kNLowRates; ++r) {
            if (!(mine >> r & 1u)) continue;
            const int dch = ((adv[r] * (t + 1)) >> 4) - ((adv[r] * t) >> 4);
            sb[r] += dch; if (sb[r] >= cap[r]) sb[r] -= cap[r];
          }
        }
        if (!RT && ((e - 1u) & 1u) == which) {          // the owner of the unit's last tile, once the other thread's last tile is done too
          if (t1 - t0 >= 2) mbar_wait(acc_full_u + 8u * ((e - 2u) & (NACC - 1)), ((e - 2u) / NACC) & 1u);
          commit2(unit_done_u, 3);
        }
      }
      TRACE_END(1, 3 + 3 * (int)which, mine_n);
    }
  } else if (warp >= 8 && warp < 16) {
    // ===== epilogue.  16x256b TMEM loads: thread T of a warp holds, for lanes l = T / 4 (cosine row of a template) and
    // l + 8 (its sine row, see r16_lane), the columns 8 i + 2 (T % 4) + {0, 1}: |rho|^2 without any cross-lane traffic.
    // Two GROUPS of four warps (one per TMEM lane quarter) take alternate tiles -- group = parity of the ABSOLUTE tile index,
    // so that the result does not depend on how the stream was cut into chunks -- and a warp walks the tile's two column
    // halves with two loads each (h = 0, 1: lanes 0-15 / 16-31 of its quarter).  With all eight warps on every tile they
    // all sat through the same barrier and TMEM-load latencies together (issue slots 21 % used); now one group computes
    // while the other waits.  The maximum of 16 |rho|^2 is found with the column index packed into the 4 low mantissa bits
    // (15 - j: the lowest column wins a tie; the truncation is 2^-19 relative), 15 integer maxima and a 4-level select tree.
    // Each group keeps a running maximum per template over its tiles of a granule and writes its own record
    // (slot 2 granule + group); the merge kernel takes the larger one, the earlier sample on a tie. =====
    const int q = warp & 3, wg = (warp - 8) >> 2, tq = lane >> 2, tc = lane & 3;
    const uint32_t acc_empty_leader = smem_u32(&bars.acc_empty[0]) & kLeaderMask;
    uint32_t e = 0;
    TRACE_BEGIN();
    FOR_F0_SEGMENTS(it, S, pA, pB) {
      const int t0 = it.cur.t, t1 = it.seg_end(), bdi = S.bds[it.cur.ib].bd;
      const int n_templates = a.bd[bdi].n_templates;
      const int p0 = (2 * it.cur.pb + (int)rank) * 64 + 16 * q + tq;      // template of h = 0; h = 1: + 8
      if constexpr (RT) {
        // Every MMA that read the old R must be complete: the previous unit's last two tiles.  One of them was this group's
        // (drained); the other group's is waited for here as an observer (its accumulator cannot be reused before r_ready).
        if (e > 1) mbar_wait(acc_full_u + 8u * ((e - 2u) & (NACC - 1)), ((e - 2u) / NACC) & 1u);
        if (e > 0) mbar_wait(acc_full_u + 8u * ((e - 1u) & (NACC - 1)), ((e - 1u) / NACC) & 1u);
        const BdPlan* B = a.bd + bdi;
        __syncwarp();
        load_R_tmem(a.sp, B->f0_slice, B->n_f0, 2 * it.cur.pb + (int)rank, tmem + ((uint32_t)(q * 32) << 16), q * 32 + lane, wg);
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(r_ready_u & kLeaderMask);
      }
      int g_left = gt - (int)((a0 + t0) % gt);                           // tiles to the end of the current granule (absolute grid)
      uint32_t own = (uint32_t)((a0 + t0) & 1) ^ (uint32_t)wg;            // 0: tile t is this group's
      uint32_t bqt[2] = {0u, 0u};                                       // running maximum of the granule (truncated bits)
      int bk[2] = {0, 0};
      float bre[2] = {0.f, 0.f}, bim[2] = {0.f, 0.f};
      for (int t = t0; t < t1; ++t, ++e, own ^= 1u) {
        if (own == 0u) {
          const uint32_t b = e & (NACC - 1), ph = (e / NACC) & 1u;
          TWAIT(0, acc_full_u + 8u * b, ph);
          __syncwarp();
          fence_after();
          const int kap0 = t * 128;
          const int valid = min(128, a.c - kap0);
#pragma unroll 1
          for (int ch = 0; ch < 2; ++ch) {                                  // column halves [0, 64), [64, 128)
            const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + b * 128u + (uint32_t)(64 * ch);
            const int cthr = 64 * ch + 2 * tc;                              // column of (i = 0, e = 0)
            uint32_t rr[2][32];
            __syncwarp();                                                   // tcgen05.ld is .aligned: the lanes may have diverged above
            tmem_ld_16x256b_x8(taddr, rr[0]);
            tmem_ld_16x256b_x8(taddr + (16u << 16), rr[1]);
            tmem_ld_wait();
            if (ch == 1) {                                                  // the whole tile is in registers or done: free the accumulator
              fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(acc_empty_leader + 8u * b);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              uint32_t (&r)[32] = rr[h];
              if constexpr (CAPTURE) {
                const int p = p0 + 8 * h;
                if (a.cap.bd == bdi && 2 * p + 1 < a.cap.rows) {
#pragma unroll
                  for (int j = 0; j < 16; ++j) {
                    const int col = cthr + 8 * (j >> 1) + (j & 1);
                    const long long k = a.k_a + kap0 + col;
                    if (col < valid && k >= a.cap.k_begin && k < a.cap.k_begin + a.cap.n) {
                      a.cap.snr[(size_t)(2 * p) * a.cap.n + (k - a.cap.k_begin)] = __uint_as_float(r[4 * (j >> 1) + (j & 1)]);
                      a.cap.snr[(size_t)(2 * p + 1) * a.cap.n + (k - a.cap.k_begin)] = __uint_as_float(r[4 * (j >> 1) + 2 + (j & 1)]);
                    }
                  }
                }
              }
#ifdef LLOID_TRACE_BUILD
              if (g_exp & 4) continue;
#endif
              uint32_t code[16];
#pragma unroll
              for (int i = 0; i < 8; ++i) {                                 // two columns per packed instruction: q = fma(re, re, im * im)
                uint64_t re2, im2, q2;
                asm("mov.b64 %0, {%1, %2};" : "=l"(re2) : "r"(r[4 * i]), "r"(r[4 * i + 1]));
                asm("mov.b64 %0, {%1, %2};" : "=l"(im2) : "r"(r[4 * i + 2]), "r"(r[4 * i + 3]));
                asm("mul.rn.f32x2 %0, %1, %1;" : "=l"(q2) : "l"(im2));
                asm("fma.rn.f32x2 %0, %1, %1, %0;" : "+l"(q2) : "l"(re2));
                asm("mov.b64 {%0, %1}, %2;" : "=r"(code[2 * i]), "=r"(code[2 * i + 1]) : "l"(q2));
              }
              if (valid < 128) {
#pragma unroll
                for (int j = 0; j < 16; ++j) if (cthr + 8 * (j >> 1) + (j & 1) >= valid) code[j] = 0u;
              }
              // Gate: only a value above the threshold can become a trigger, and only one above the granule's running
              // maximum changes it.  The plain maximum of the 16 |rho|^2 (8 instructions) against max(theta^2 (1 - 2^-16),
              // running maximum) decides for the whole warp whether the index bookkeeping below (pack, 15 maxima, select
              // tree: 80 of the 150 instructions per half tile) runs at all; at theta = 4 in noise it does for one warp in
              // six.  A granule without any value above the threshold leaves a record with q = 0, which the merge kernel
              // never turns into a trigger.
              {
                uint32_t mx = max(max(code[0], code[1]), code[2]);
#pragma unroll
                for (int j = 3; j < 15; j += 2) mx = max(max(mx, code[j]), code[j + 1]);
                mx = max(mx, code[15]);
                if (!__any_sync(0xffffffffu, mx > max(a.q_gate, bqt[h]))) continue;
              }
#pragma unroll
              for (int j = 0; j < 16; ++j) code[j] = (code[j] & ~15u) | (uint32_t)(15 - j);
#pragma unroll
              for (int st = 8; st >= 1; st >>= 1)
#pragma unroll
                for (int j = 0; j < st; ++j) code[j] = max(code[j], code[j + st]);
              const uint32_t m = code[0];
              const int jw = 15 - (int)(m & 15u);
              // select tree on the bits of jw: e = jw & 1, i = jw >> 1
              uint32_t sr[8], si[8];
#pragma unroll
              for (int i = 0; i < 8; ++i) { sr[i] = (jw & 1) ? r[4 * i + 1] : r[4 * i]; si[i] = (jw & 1) ? r[4 * i + 3] : r[4 * i + 2]; }
#pragma unroll
              for (int i = 0; i < 4; ++i) { sr[i] = (jw & 2) ? sr[2 * i + 1] : sr[2 * i]; si[i] = (jw & 2) ? si[2 * i + 1] : si[2 * i]; }
#pragma unroll
              for (int i = 0; i < 2; ++i) { sr[i] = (jw & 4) ? sr[2 * i + 1] : sr[2 * i]; si[i] = (jw & 4) ? si[2 * i + 1] : si[2 * i]; }
              const uint32_t wr = (jw & 8) ? sr[1] : sr[0], wi = (jw & 8) ? si[1] : si[0];
              if ((m & ~15u) > bqt[h]) {                                    // later columns and later tiles never win ties
                bqt[h] = m & ~15u; bk[h] = kap0 + cthr + 8 * (jw >> 1) + (jw & 1);
                bre[h] = __uint_as_float(wr); bim[h] = __uint_as_float(wi);
              }
            }
          }
        }
        // granule end (reached by both groups, whether or not the last tile was theirs): merge the 4 threads of a template,
        // write this group's record -- also when it saw no tile or no value above the gate (q = 0)
        if (t + 1 == t1 || --g_left == 0) {                                // (no 64-bit division per tile: a countdown)
          g_left = gt;
          const int gi = (int)((a0 + t) / gt - a0 / gt);
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            float bq = fmaf(bre[h], bre[h], bim[h] * bim[h]);
            int k = bk[h];
            float re = bre[h], im = bim[h];
#pragma unroll
            for (int x = 1; x <= 2; x <<= 1) {
              const float oq = __shfl_xor_sync(0xffffffffu, bq, x), ore = __shfl_xor_sync(0xffffffffu, re, x), oim = __shfl_xor_sync(0xffffffffu, im, x);
              const int ok = __shfl_xor_sync(0xffffffffu, k, x);
              if (oq > bq || (oq == bq && ok < k)) { bq = oq; k = ok; re = ore; im = oim; }
            }
            const int p = p0 + 8 * h;
            if (tc == 0 && p < n_templates) {
              Peak pk; pk.q = bq; pk.kappa = k; pk.re = re; pk.im = im;
              a.partials[((size_t)bdi * a.slots_cap + 2 * gi + wg) * a.max_templates + p] = pk;
            }
            bqt[h] = 0u; bk[h] = 0; bre[h] = 0.f; bim[h] = 0.f;
          }
        }
      }
    }
    if (rank == 0 && tid == 256) TRACE_END(1, 4, (int)e);
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
  pl->n_tab = 0;
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
    for (int v = 0; v < 4; ++v) { U.n_items[v] = 0; U.tab_off[v] = 0; }
    for (int v = 0; v < U.n_var; ++v) {
      const int mis = v * U.adv;
      const int nch = (mis + U.adv + 2 * kKUp + 15) / 16;
      if (nch > cap) return true;
      struct Item { uint32_t idesc, p_lo, d_col; int ch; };
      std::vector<Item> items;
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
        Item it;
        it.idesc = (1u << 4) | ((uint32_t)(nn >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
        it.p_lo = (uint32_t)((base * sizeof(__half)) >> 4) | ((uint32_t)half << 16);     // LBO = half * 16 bytes
        it.d_col = (uint32_t)n0;
        it.ch = ch;
        items.push_back(it);
      }
      U.n_items[v] = (int)items.size();
      U.tab_off[v] = pl->n_tab;
      if (pl->n_tab + cap * (int)items.size() > kPairTabMax) return true;
      for (int s0 = 0; s0 < cap; ++s0)
        for (const Item& it : items) {
          PairMma& m = pl->tab[pl->n_tab++];
          m.a_off = (uint32_t)((s0 + it.ch) % cap) * 256u; m.p_lo = it.p_lo; m.idesc = it.idesc; m.d_col = it.d_col;
        }
    }
  }
  pl->p_bytes = (int)((pblob[0].size() * sizeof(__half) + 127) / 128 * 128);
  pl->q_bytes = q_bytes;

  // Where the stationary R of a unit lives (template parameter RT of the kernels).  In shared memory it competes with P, the
  // windows and >= 3 y stages: if EVERY (bin, detector) fits that way the bank runs the RT = false kernels; otherwise the
  // whole bank runs the RT = true kernels (R in TMEM, K <= 512), and only what exceeds THAT is left to the FFMA kernels.
  {
    const int lim_f0_smem = (PK_SMEM_BUDGET - pl->p_bytes - pl->q_bytes - 3 * 16384) / 256;
    const int lim_low_smem = (PK_SMEM_BUDGET - 3 * 16384) / 256;
    bool rt = false;
    for (int b = 0; b < n_bd; ++b) {
      if (pl->excluded[b]) continue;
      if (pl->bd_host[b].l_sum > lim_f0_smem) rt = true;
      for (int r = 0; r < pl->n_lr; ++r) if (pl->groups_host[(size_t)b * pl->n_lr + r].l_sum > lim_low_smem) rt = true;
    }
    if (getenv("LLOID_R_TMEM")) rt = atoi(getenv("LLOID_R_TMEM")) != 0;      // debugging / A-B measurements
    pl->r_tmem = rt;
    const int lim_f0 = rt ? PK_KMAX : lim_f0_smem, lim_low = rt ? PK_KMAX : lim_low_smem;
    if (rt && PK_SMEM_BUDGET - pl->p_bytes - pl->q_bytes < 3 * 16384) return true;
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
  const int f0_fixed = (pl->r_tmem ? 0 : pl->l_sum_f0_max * 256) + pl->p_bytes + pl->q_bytes;
  const int low_fixed = pl->r_tmem ? 0 : pl->l_sum_low_max * 256;
  // y stage slot: the largest stage of any unit the kernel streams (a unit with nm = sum L_pad / 16 MMAs per tile is cut
  // into ceil(nm / ycap) stages of ceil(nm / stages) MMAs at most, 2 KB per MMA and CTA)
  // (with R in shared memory the ring is short -- 3 slots of 14 KB at config 2 -- and stages of <= 6 MMAs = 4 slots of 10 KB
  // measured 4 % faster in the f0 kernel; with R in TMEM the ring is long and <= 8 is as good or better)
  pl->ycap = getenv("LLOID_YCAP") ? std::max(2, std::min(16, atoi(getenv("LLOID_YCAP")))) : (pl->r_tmem ? 8 : 6);
  int ys_f0 = 2048, ys_low = 2048;
  auto stage_bytes = [&](int l_sum) { const int nm = l_sum / 16, nst = stage_count(nm, pl->ycap); return (nm + nst - 1) / nst * 2048; };
  for (int b = 0; b < n_bd; ++b) {
    if (pl->excluded[b]) continue;
    ys_f0 = std::max(ys_f0, stage_bytes(pl->bd_host[b].l_sum));
    for (int r = 0; r < pl->n_lr; ++r) {
      const RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + r];
      if (G.n_slices) ys_low = std::max(ys_low, stage_bytes(G.l_sum));
    }
  }
  pl->f0_ystage = ys_f0; pl->low_ystage = ys_low;
  pl->f0_stages = std::min(PK_NSY_MAX, (PK_SMEM_BUDGET - f0_fixed) / ys_f0);
  pl->low_stages = std::min(PK_NSY_MAX, (PK_SMEM_BUDGET - low_fixed) / ys_low);
  pl->f0_smem = f0_fixed + pl->f0_stages * ys_f0;
  pl->low_smem = low_fixed + pl->low_stages * ys_low;
  if (getenv("LLOID_PLAN_PRINT"))
    fprintf(stderr, "[lloid plan] r_tmem %d  f0: R %d B, P %d B, Q windows %d B, %d y slots of %d B   low: R %d B, %d y slots of %d B   ycap %d\n",
            (int)pl->r_tmem, pl->l_sum_f0_max * 256, pl->p_bytes, pl->q_bytes, pl->f0_stages, ys_f0, pl->l_sum_low_max * 256, pl->low_stages, ys_low, pl->ycap);
  // device tables
  std::vector<LowUnit> units;                             // rate-major: all units of a rate have the same tile count
  std::vector<SchedBd> low_cells;                         // low-rate schedule: per class one entry per group (LowSched)
  // rho^(d) buffers: ONE allocation (chunk-local: a part of a split bank takes it from the parent's shared set)
  size_t q_total = 0;
  for (int r = 0; r < pl->n_lr; ++r)
    for (int b = 0; b < n_bd; ++b) {
      const RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + r];
      if (G.n_slices && !pl->excluded[b]) q_total += (size_t)G.n_rb * 2 * G.q_groups_cap * 2048;
    }
  uint8_t* q_base = nullptr;
  if (q_total) {
    if (pl->q_alloc) {
      q_base = (uint8_t*)pl->q_alloc(pl->q_ctx, q_total);
      if (!q_base) { snprintf(err, errlen, "fp16 plan: %zu bytes for the low-rate SNR buffers could not be allocated", q_total); return false; }
    } else {
      void* q = nullptr;
      if (!plan_alloc(pl, &q, q_total, true, bytes, err, errlen)) return false;
      q_base = (uint8_t*)q;
    }
  }
  size_t q_off = 0;
  for (int r = 0; r < pl->n_lr; ++r) {
    pl->units_per_rate[r] = 0; pl->low_wsum[r] = 0; pl->low_cells_per_rate[r] = 0;
    for (int b = 0; b < n_bd; ++b) {
      RateGroup& G = pl->groups_host[(size_t)b * pl->n_lr + r];
      if (G.n_slices == 0 || pl->excluded[b]) continue;
      G.Q = (__half*)(q_base + q_off);
      q_off += (size_t)G.n_rb * 2 * G.q_groups_cap * 2048;
      {
        SchedBd e; e.bd = (int32_t)units.size(); e.n_pb = G.n_rb; e.w = G.l_sum / 16; e.pad = 0; e.cum = pl->low_wsum[r];
        low_cells.push_back(e);
        pl->low_wsum[r] += (long long)G.n_rb * e.w;
        ++pl->low_cells_per_rate[r];
      }
      for (int rb = 0; rb < G.n_rb; ++rb) units.push_back(LowUnit{b * pl->n_lr + r, rb});
      pl->units_per_rate[r] += G.n_rb;
    }
  }
  // f0 schedule entries: one per tensor-path (bin, detector); cost per tile and template block = MMAs: K / 16 of the
  // d == 1 slices + interpolation chunks
  std::vector<SchedBd> f0_sched;
  pl->f0_wsum = 0;
  for (int b = 0; b < n_bd; ++b) {
    if (pl->excluded[b]) continue;
    int w = pl->bd_host[b].l_sum / 16;
    for (int r = 0; r < pl->n_lr; ++r) {
      if (pl->groups_host[(size_t)b * pl->n_lr + r].n_slices == 0) continue;
      w += pl->rate[r].n_items[0];
    }
    SchedBd e; e.bd = b; e.n_pb = pl->bd_host[b].n_rb; e.w = w; e.pad = 0; e.cum = pl->f0_wsum;
    f0_sched.push_back(e);
    pl->f0_wsum += (long long)e.n_pb * w;
  }
  pl->f0_n_bds = (int)f0_sched.size();
  pl->f0_n_pb = f0_sched.empty() ? 0 : f0_sched[0].n_pb;                 // template blocks per (bin, detector) if uniform, else 0
  for (const SchedBd& e : f0_sched) if (e.n_pb != pl->f0_n_pb) pl->f0_n_pb = 0;
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
  if (!upload((void**)&pl->low_cells_dev, low_cells.data(), low_cells.size() * sizeof(SchedBd))) return false;
  if (!upload((void**)&pl->f0_sched_dev, f0_sched.data(), f0_sched.size() * sizeof(SchedBd))) return false;

  // opt-in shared memory: the architecture maximum, for every kernel of this file, on this device (never lowered
  // by a later, smaller bank)
  cudaError_t e = set_max_dyn_smem(f0_pair_kernel<false, false>);
  if (e == cudaSuccess) e = set_max_dyn_smem(f0_pair_kernel<true, false>);
  if (e == cudaSuccess) e = set_max_dyn_smem(f0_pair_kernel<false, true>);
  if (e == cudaSuccess) e = set_max_dyn_smem(f0_pair_kernel<true, true>);
  if (e == cudaSuccess) e = set_max_dyn_smem(lowrate_pair_kernel<false>);
  if (e == cudaSuccess) e = set_max_dyn_smem(lowrate_pair_kernel<true>);
  if (e != cudaSuccess) { snprintf(err, errlen, "fp16 plan: cudaFuncSetAttribute failed: %s", cudaGetErrorString(e)); return false; }
  pl->tensor_recon = true;
  return true;
}

bool f16_plan_tensor_recon(const F16Plan* pl) { return pl && pl->tensor_recon; }
bool f16_plan_r_tmem(const F16Plan* pl) { return pl && pl->tensor_recon && pl->r_tmem; }
void f16_plan_disable_tensor_recon(F16Plan* pl) { if (pl) pl->tensor_recon = false; }
const uint8_t* f16_plan_excluded(const F16Plan* pl) { return (pl && pl->tensor_recon && pl->any_excluded) ? pl->excluded.data() : nullptr; }

int f16_read_trace(long long* out, int reset)
{
  if (cudaMemcpyFromSymbol(out, g_trace, sizeof(long long) * 128) != cudaSuccess) return 1;
  if (reset) { static long long z[128]; cudaMemcpyToSymbol(g_trace, z, sizeof z); }
  return 0;
}

int f16_granule_tiles(int peak_window)
{
  int gt = peak_window / kTimeTile;
  while (gt > 32 && gt % 2 == 0) gt /= 2;
  return gt < 1 ? 1 : gt;
}

int launch_recon_f16(F16Plan* pl, const SliceParams* sp_dev, Peak* partials, int slots_cap, int max_templates,
                     int c, int64_t k_a, int gt, float theta, Capture cap, cudaStream_t st, int64_t* launches, cudaEvent_t after_lowrate)
{
  const int n_clusters = std::max(1, pl->n_sm / 2);
#ifdef LLOID_TRACE_BUILD
  { const int exp_bits = getenv("LLOID_EXP") ? atoi(getenv("LLOID_EXP")) : 0; cudaMemcpyToSymbol(g_exp, &exp_bits, sizeof(int)); }
#endif
  if (pl->low_units > 0) {
    LowPArgs la;
    memset(&la, 0, sizeof la);
    la.sp = sp_dev; la.groups = pl->groups_dev; la.units = (const LowUnit*)pl->units_dev;
    la.r_bytes = pl->l_sum_low_max * 256; la.nsy = pl->low_stages; la.ystage = pl->low_ystage; la.ycap = pl->ycap; la.trace = getenv("LLOID_TRACE") ? 1 : 0;
    LowSched& sc = la.sched;
    sc.cells = pl->low_cells_dev; sc.n_cls = pl->n_lr;
    long long tiles_total = 0;
    for (int r = 0; r < pl->n_lr; ++r) {
      sc.cell_begin[r + 1] = sc.cell_begin[r] + pl->low_cells_per_rate[r];
      sc.n_tiles[r] = (((c >> pl->rate[r].log2d) + 2 * kKUp) + 127) / 128;
      sc.total[r] = pl->low_wsum[r];
      sc.base[r + 1] = sc.base[r] + pl->low_wsum[r] * sc.n_tiles[r];
      tiles_total += (long long)sc.n_tiles[r] * pl->units_per_rate[r];
    }
    for (int r = 0; r < pl->n_lr; ++r) {
      // time block of class r = the tiles one cluster gets through in its share of the cost (mean cost per tile of the class)
      const long long share = (sc.base[pl->n_lr] + n_clusters - 1) / n_clusters;
      const long long w_mean = pl->units_per_rate[r] ? std::max<long long>(1, pl->low_wsum[r] / pl->units_per_rate[r]) : 1;
      long long gb = getenv("LLOID_LOW_BLOCK") ? atoi(getenv("LLOID_LOW_BLOCK")) : share / w_mean;
      sc.gb[r] = (int)std::max<long long>(1, std::min<long long>(gb, sc.n_tiles[r]));
    }
    const int grid = 2 * (int)std::min<long long>(n_clusters, tiles_total);
    if (pl->r_tmem) lowrate_pair_kernel<true><<<grid, PK_THREADS, pl->low_smem, st>>>(la);
    else lowrate_pair_kernel<false><<<grid, PK_THREADS, pl->low_smem, st>>>(la);
    ++*launches;
  }
  if (after_lowrate) cudaEventRecord(after_lowrate, st);
  if (getenv("LLOID_DEBUG_SYNC") && cudaStreamSynchronize(st) != cudaSuccess) { fprintf(stderr, "lloid: lowrate_pair_kernel faulted\n"); return 1; }
  F0PArgs a;
  memset(&a, 0, sizeof a);
  a.sp = sp_dev; a.bd = pl->bd_dev; a.groups = pl->groups_dev;
  a.P = reinterpret_cast<const uint8_t*>(pl->p_dev);
  a.partials = partials; a.cap = cap; a.k_a = k_a;
  a.n_lr = pl->n_lr; a.c = c; a.r_bytes = pl->l_sum_f0_max * 256; a.p_bytes = pl->p_bytes; a.q_bytes = pl->q_bytes;
  a.nsy = pl->f0_stages; a.ystage = pl->f0_ystage; a.ycap = pl->ycap; a.slots_cap = slots_cap; a.max_templates = max_templates;
  a.trace = getenv("LLOID_TRACE") ? 1 : 0;
  const int n_tiles = (c + 127) / 128;
  a.sched.bds = pl->f0_sched_dev; a.sched.n_bds = pl->f0_n_bds; a.sched.n_tiles = n_tiles;
  // Time block = one cluster's share of the tiles, rounded up to whole granules: cluster i then works on (about) the i-th
  // (time block, template block) cell, so the clusters that walk the template blocks of one time block start together
  // and read the same y tiles within a few tiles of each other: 7 of the 8 reads of a y tile hit L2.  (With fixed blocks
  // of 64 tiles a cluster walked 3.5 cells, a y tile was re-read 64 tiles = 0.1 ms later, long after L2 had turned over:
  // 1.87 GB of DRAM reads per config-2 launch for 0.67 GB of operands.)
  {
    const long long all_tiles = (long long)pl->combos_host.size() * n_tiles;
    long long gb = getenv("LLOID_F0_BLOCK") ? atoi(getenv("LLOID_F0_BLOCK")) : (all_tiles + n_clusters - 1) / n_clusters;
    gb = std::max<long long>(gt, (gb + gt - 1) / gt * gt);
    a.sched.gt = gt; a.sched.gb = (int)std::min<long long>(gb, (long long)(n_tiles + gt - 1) / gt * gt + gt);
  }
  a.sched.total = pl->f0_wsum; a.sched.a0 = k_a / kTimeTile;
  a.sched.n_pb = getenv("LLOID_F0_ORDER_PB") ? pl->f0_n_pb : 0;          // template-block-major order: measured, no gain (see F0Sched)
  {
    const float g = theta * theta * (1.0f - 1.0f / 65536.0f);
    a.q_gate = getenv("LLOID_NO_GATE") ? 0u : *reinterpret_cast<const uint32_t*>(&g);
  }
  for (int r = 0; r < kNLowRates; ++r) a.rate[r] = pl->rate[r];
  memcpy(a.tab, pl->tab, sizeof a.tab);
  const long long pair_tiles = (long long)pl->combos_host.size() * n_tiles;
  const int grid = 2 * (int)std::min<long long>(n_clusters, pair_tiles);
  if (pl->r_tmem) {
    if (cap.snr) f0_pair_kernel<true, true><<<grid, PK_THREADS, pl->f0_smem, st>>>(a);
    else f0_pair_kernel<false, true><<<grid, PK_THREADS, pl->f0_smem, st>>>(a);
  } else {
    if (cap.snr) f0_pair_kernel<true, false><<<grid, PK_THREADS, pl->f0_smem, st>>>(a);
    else f0_pair_kernel<false, false><<<grid, PK_THREADS, pl->f0_smem, st>>>(a);
  }
  ++*launches;
  const cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) fprintf(stderr, "lloid: f0_pair_kernel launch (grid %d, %d threads, %d B shared, %zu B params): %s\n", grid, PK_THREADS, pl->f0_smem, sizeof a, cudaGetErrorString(e));
  return e == cudaSuccess ? 0 : 1;
}

}  // namespace lloid
