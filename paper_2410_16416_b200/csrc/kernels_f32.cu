// fp32 path (LLOID_F32): A2 basis FIR and A3+A4+A5 reconstruction / upsample-accumulate / |rho|^2 /
// windowed max on the CUDA cores (FFMA).  TF32 tensor MMAs keep a 10-bit mantissa and cannot meet the
// 1e-3 absolute SNR parity of BASELINE.json's fp32 path, so this path is plain fp32.
// The fp16 tensor-core path lives in kernels_f16.cu.
#include "lloid_internal.h"

#include <algorithm>

namespace lloid {

// Packed fp32 FMA (FFMA2 on sm_100a): two independent fma.rn.f32 per instruction, bit-identical to the scalar form.
// The FMA pipe runs it at the same flop rate, but it needs half the issue slots -- the register-tiled kernels below
// were issue-bound (71 % issue-active, FFMA only 78 % of the instructions).  ptxas folds pack2(a, a) into a scalar
// broadcast operand (R4.F32), so the duplicated multiplicand costs nothing.
typedef unsigned long long u64;
__device__ __forceinline__ u64 pack2(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ void ffma2(u64& c, u64 a, u64 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b)); }

// Eight consecutive l of one reconstruction row i / one y row r, from the fp32 row-major arrays or (PK: the fp16
// path's CUDA-core fallback for banks the tensor reconstruction cannot hold) from the packed fp16 operands, where the
// same eight values are one 16-byte core-matrix row:  R16[i / 128][l / 8][r16_lane(i % 128)][l % 8],
// Y16[r / 64][slice of the rate group][l / 8][r % 64][l % 8] (y_step64 bytes per 64-row tile).  l is a multiple of 8.
__device__ __forceinline__ void h8_to_f(const uint4 v, float4& lo, float4& hi)
{
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&v.x)), b = __half22float2(*reinterpret_cast<const __half2*>(&v.y));
  const float2 c = __half22float2(*reinterpret_cast<const __half2*>(&v.z)), d = __half22float2(*reinterpret_cast<const __half2*>(&v.w));
  lo = make_float4(a.x, a.y, b.x, b.y); hi = make_float4(c.x, c.y, d.x, d.y);
}
// base address of (row i, l) / (y row r, l) and the byte step per 8 l: both layouts are linear in l / 8
template <bool PK>
__device__ __forceinline__ const char* base8_R(const SliceParams& P, int i, int l, int& step)
{
  if constexpr (PK) {
    step = 128 * 8 * 2;
    return reinterpret_cast<const char*>(P.R16 + (((size_t)(i >> 7) * (P.L_pad >> 3) + (l >> 3)) * 128 + r16_lane(i & 127)) * 8);
  } else {
    step = 32;
    return reinterpret_cast<const char*>(P.R32 + (size_t)i * P.L_pad + l);
  }
}
template <bool PK>
__device__ __forceinline__ const char* base8_Y(const SliceParams& P, int r, int l, int& step)
{
  if constexpr (PK) {
    step = 64 * 8 * 2;
    return reinterpret_cast<const char*>(P.Y) + (size_t)(r >> 6) * P.y_step64 + (((size_t)(l >> 3)) * 64 + (r & 63)) * 16;
  } else {
    step = 32;
    return reinterpret_cast<const char*>(reinterpret_cast<const float*>(P.Y) + (size_t)r * P.L_pad + l);
  }
}
template <bool PK, bool NC>
__device__ __forceinline__ void load8(const char* p, float4& lo, float4& hi)
{
  if constexpr (PK) {
    h8_to_f(NC ? __ldg(reinterpret_cast<const uint4*>(p)) : *reinterpret_cast<const uint4*>(p), lo, hi);
  } else {
    const float4* q = reinterpret_cast<const float4*>(p);
    lo = NC ? __ldg(q) : q[0]; hi = NC ? __ldg(q + 1) : q[1];
  }
}


// ------------------------------------------------------------------------------------------------
// A2  y^s_l[j] = sum_t U^s[l,t] x^s[j - n_s + t]                     ("cross-correlates")
//
// CTA tile: 128 low-rate outputs x 32 basis filters, 128 threads, thread tile 8 (time) x 4 (l).
// The strain window of the tile (128 + n_s samples) is staged once in shared memory; U streams
// through in 64-tap chunks, transposed to [t][l].  Per 8 taps a thread reads a 16-sample strain
// window (4 LDS.128) and 8 float4 of U, and issues 256 FMAs: the Toeplitz operand is never
// materialised anywhere.
// ------------------------------------------------------------------------------------------------
constexpr int FIR_TM = 128, FIR_TL = 32, FIR_KC = 64, FIR_US = 36;

__global__ void __launch_bounds__(128)
fir_f32_kernel(const SliceParams* __restrict__ sp, const RateParams* __restrict__ rates, int o, int c, int zs_len)
{
  const SliceParams P = sp[blockIdx.z];
  const int rows_needed = (P.d == 1) ? c : (c >> P.log2d) + 2 * kKUp;
  const int r0 = blockIdx.x * FIR_TM;
  const int l0 = blockIdx.y * FIR_TL;
  if (r0 >= rows_needed || l0 >= P.L_pad) return;

  extern __shared__ __align__(16) float smem_f[];
  float* zs = smem_f;                 // [zs_len]
  float* Us = smem_f + zs_len;        // [FIR_KC][FIR_US]
  const RateParams R = rates[P.rate_idx];
  const float* __restrict__ xs = R.xs32 + (size_t)P.det * R.xs_len;
  const int tid = threadIdx.x;
  const int n_taps = P.n_taps;
  const int jj_start = P.jjY0 + (o >> P.log2d) + r0 - n_taps;
  for (int i = tid; i < zs_len; i += 128) {
    const int idx = jj_start + i;
    zs[i] = (i < FIR_TM + n_taps && idx >= 0 && idx < R.xs_len) ? xs[idx] : 0.f;
  }

  const int tl = tid & 7, tj = tid >> 3;
  u64 acc[8][2];                      // [time row][basis pair], packed fp32 x 2
#pragma unroll
  for (int j = 0; j < 8; ++j) { acc[j][0] = acc[j][1] = 0ull; }

  const float* __restrict__ U = P.U32;
  for (int t0 = 0; t0 < n_taps; t0 += FIR_KC) {
    __syncthreads();
#pragma unroll 4
    for (int i = 0; i < (FIR_KC * FIR_TL) / 128; ++i) {
      const int e = tid + 128 * i;
      const int ll = e / FIR_KC, tt = e % FIR_KC;
      const int t = t0 + tt;
      Us[tt * FIR_US + ll] = (t < n_taps) ? __ldg(U + (size_t)(l0 + ll) * n_taps + t) : 0.f;
    }
    __syncthreads();
#pragma unroll 2
    for (int tt8 = 0; tt8 < FIR_KC; tt8 += 8) {
      float zw[16];
      const float4* zp = reinterpret_cast<const float4*>(zs + tj * 8 + t0 + tt8);
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float4 q = zp[v];
        zw[4 * v] = q.x; zw[4 * v + 1] = q.y; zw[4 * v + 2] = q.z; zw[4 * v + 3] = q.w;
      }
#pragma unroll
      for (int tt = 0; tt < 8; ++tt) {
        const float4 u = *reinterpret_cast<const float4*>(Us + (tt8 + tt) * FIR_US + tl * 4);
        const u64 u01 = pack2(u.x, u.y), u23 = pack2(u.z, u.w);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const u64 zz = pack2(zw[j + tt], zw[j + tt]);
          ffma2(acc[j][0], zz, u01);
          ffma2(acc[j][1], zz, u23);
        }
      }
    }
  }
  float* Y = reinterpret_cast<float*>(P.Y);
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const int r = r0 + tj * 8 + j;
    float4 v;
    unpack2(acc[j][0], v.x, v.y); unpack2(acc[j][1], v.z, v.w);
    if (r < P.y_rows_cap) *reinterpret_cast<float4*>(Y + (size_t)r * P.L_pad + l0 + tl * 4) = v;
  }
}

void launch_fir_f32(const SliceParams* sp_dev, const SliceParams* sp_host, int n_problems,
                    const RateParams* rates_dev, int n_det, int o, int c, cudaStream_t st, int64_t* launches)
{
  (void)n_det;
  int max_rows = 0, max_lt = 0, max_taps = 0;
  for (int i = 0; i < n_problems; ++i) {
    const SliceParams& P = sp_host[i];
    const int rows = (P.d == 1) ? c : (c >> P.log2d) + 2 * kKUp;
    if (rows > max_rows) max_rows = rows;
    if (P.L_pad / FIR_TL > max_lt) max_lt = P.L_pad / FIR_TL;
    if (P.n_taps > max_taps) max_taps = P.n_taps;
  }
  const int zs_len = FIR_TM + ((max_taps + FIR_KC - 1) / FIR_KC) * FIR_KC + 16;
  const size_t smem = sizeof(float) * ((size_t)zs_len + FIR_KC * FIR_US);
  dim3 grid((max_rows + FIR_TM - 1) / FIR_TM, max_lt, n_problems);
  fir_f32_kernel<<<grid, 128, smem, st>>>(sp_dev, rates_dev, o, c, zs_len);
  ++*launches;
}

// ------------------------------------------------------------------------------------------------
// A3 + A4 + A5 fused:  rho^s = R^s y^s at the slice rate, interpolated to f0 and summed over slices
// in registers, then |rho|^2 and the per-template maximum of the tile.  The dense SNR never leaves
// the SM (the SNR series is too large to move; here it is not even written to HBM).
//
// CTA tile: 64 real rows (32 templates) x 128 f0 samples, 256 threads as 16 (row groups of 4) x
// 16 (column groups of 8); each thread keeps a 4 x 8 fp32 accumulator of the f0-rate SNR.
// Per slice: a K-chunked SGEMM R^s[64 x L] * y^s[L x Ks] with Ks = 128 (d = 1, accumulated
// directly) or 128/d + 16 low-rate samples (d > 1, staged through shared memory and interpolated
// with the 16-tap polyphase weights w_phi[i] = d lp[d i + phi]).
// ------------------------------------------------------------------------------------------------
constexpr int RC_RT = 64, RC_CT = kTimeTile, RC_KC = 32, RC_RS = RC_RT + 4, RC_YS = RC_CT + 4;
constexpr int RC_KSMAX = RC_CT / 2 + 2 * kKUp;   // 80 low-rate samples at d = 2
constexpr int RC_RHO_S = RC_KSMAX + 1;

template <int D, int NR>
__device__ __forceinline__ void upsample_acc(float (&acc)[NR][8], const float* __restrict__ rho,
                                             const float* __restrict__ wsm, int ty, int tx)
{
  // thread tile: rows NR ty + r, columns kl = 8 tx + cc;  low-rate local index ml = kl / D, phase phi = kl % D
  // c[kl] += sum_{i=-8}^{7} wsm[(i+8)*32 + phi] * rho[row][ml + 8 - i]
  if constexpr (D >= 8) {
    const int ml = (8 * tx) / D;
    const int phi0 = (8 * tx) % D;
#pragma unroll
    for (int i = -kKUp; i < kKUp; ++i) {
      const float4 w0 = *reinterpret_cast<const float4*>(wsm + (i + kKUp) * 32 + phi0);
      const float4 w1 = *reinterpret_cast<const float4*>(wsm + (i + kKUp) * 32 + phi0 + 4);
#pragma unroll
      for (int r = 0; r < NR; ++r) {
        const float v = rho[(NR * ty + r) * RC_RHO_S + ml + kKUp - i];
        acc[r][0] = fmaf(w0.x, v, acc[r][0]); acc[r][1] = fmaf(w0.y, v, acc[r][1]);
        acc[r][2] = fmaf(w0.z, v, acc[r][2]); acc[r][3] = fmaf(w0.w, v, acc[r][3]);
        acc[r][4] = fmaf(w1.x, v, acc[r][4]); acc[r][5] = fmaf(w1.y, v, acc[r][5]);
        acc[r][6] = fmaf(w1.z, v, acc[r][6]); acc[r][7] = fmaf(w1.w, v, acc[r][7]);
      }
    }
  } else {
    // d = 2, 4: groups of TG taps whose TG x D weights stay in registers; per row the NM + TG - 1 low-rate samples
    // the group touches are read once (the straightforward loop reads one sample per D multiply-adds)
    constexpr int NM = 8 / D;                     // distinct low-rate indices under the 8 columns
    constexpr int TG = 16 / D;
    constexpr int NV = NM + TG - 1;
    const int ml0 = (8 * tx) / D;
#pragma unroll
    for (int g = 0; g < 2 * kKUp / TG; ++g) {     // taps i = -K_up + g TG + t
      float w[TG][D];
#pragma unroll
      for (int t = 0; t < TG; ++t)
#pragma unroll
        for (int p = 0; p < D; ++p) w[t][p] = wsm[(g * TG + t) * 32 + p];
#pragma unroll
      for (int r = 0; r < NR; ++r) {
        // sample index ml0 + m + K_up - i = (ml0 + 2 K_up - g TG - (TG - 1)) + m + (TG - 1 - t)
        const float* __restrict__ vr = rho + (NR * ty + r) * RC_RHO_S + ml0 + 2 * kKUp - g * TG - (TG - 1);
        float v[NV];
#pragma unroll
        for (int j = 0; j < NV; ++j) v[j] = vr[j];
#pragma unroll
        for (int t = 0; t < TG; ++t)
#pragma unroll
          for (int m = 0; m < NM; ++m)
#pragma unroll
            for (int p = 0; p < D; ++p) acc[r][m * D + p] = fmaf(w[t][p], v[m + TG - 1 - t], acc[r][m * D + p]);
      }
    }
  }
}

// Same interpolation on the packed accumulators of the 8 x 8 tile: acc[r][j] = columns (8 tx + 2 j, 8 tx + 2 j + 1).
// rho rows have stride RQ_RHO_S = 84 floats.  d >= 8: one sample per (tap, row); the two row groups a warp covers
// (ty, ty + 1) read the same columns, so odd row groups are stored with the column XOR 16 (disjoint banks).
// d = 2, 4: the NM + TG - 1 samples of a tap group start one past a 16-byte (d = 2) / 8-byte (d = 4) boundary; they
// are read as 3 aligned LDS.128 / LDS.64 (lane stride 16 / 8 bytes: no bank conflicts) and the first value dropped.
constexpr int RQ_RHO_S = 84;

template <int D>
__device__ __forceinline__ void upsample_acc2(u64 (&acc)[8][4], const float* __restrict__ rho,
                                              const float* __restrict__ wsm, int ty, int tx)
{
  if constexpr (D >= 8) {
    const int ml = (8 * tx) / D;
    const int phi0 = (8 * tx) % D;
    const int sw = (ty & 1) * 16;
    const float* __restrict__ rrow = rho + (8 * ty) * RQ_RHO_S;
#pragma unroll
    for (int i = -kKUp; i < kKUp; ++i) {
      const float4 w0 = *reinterpret_cast<const float4*>(wsm + (i + kKUp) * 32 + phi0);
      const float4 w1 = *reinterpret_cast<const float4*>(wsm + (i + kKUp) * 32 + phi0 + 4);
      const u64 wp[4] = {pack2(w0.x, w0.y), pack2(w0.z, w0.w), pack2(w1.x, w1.y), pack2(w1.z, w1.w)};
      const int col = (ml + kKUp - i) ^ sw;
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const float v = rrow[r * RQ_RHO_S + col];
        const u64 vv = pack2(v, v);
#pragma unroll
        for (int j = 0; j < 4; ++j) ffma2(acc[r][j], vv, wp[j]);
      }
    }
  } else {
    constexpr int NM = 8 / D, TG = 16 / D, DH = D / 2;
    constexpr int VW = (D == 2) ? 4 : 2;            // floats per aligned load; 3 loads cover the window + 1
    const int ml0 = (8 * tx) / D;
#pragma unroll
    for (int g = 0; g < 2 * kKUp / TG; ++g) {     // taps i = -K_up + g TG + t
      u64 w[TG][DH];
#pragma unroll
      for (int t = 0; t < TG; ++t)
#pragma unroll
        for (int h = 0; h < DH; ++h) {
          const float2 ww = *reinterpret_cast<const float2*>(wsm + (g * TG + t) * 32 + 2 * h);
          w[t][h] = pack2(ww.x, ww.y);
        }
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        // sample index ml0 + m + K_up - i = start + m + (TG - 1 - t), start = ml0 + 2 K_up - g TG - (TG - 1); start - 1 is aligned
        const float* __restrict__ vr = rho + (8 * ty + r) * RQ_RHO_S + ml0 + 2 * kKUp - g * TG - (TG - 1) - 1;
        float v[3 * VW];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          if constexpr (D == 2) {
            const float4 x = *reinterpret_cast<const float4*>(vr + 4 * q);
            v[4 * q] = x.x; v[4 * q + 1] = x.y; v[4 * q + 2] = x.z; v[4 * q + 3] = x.w;
          } else {
            const float2 x = *reinterpret_cast<const float2*>(vr + 2 * q);
            v[2 * q] = x.x; v[2 * q + 1] = x.y;
          }
        }
#pragma unroll
        for (int t = 0; t < TG; ++t)
#pragma unroll
          for (int m = 0; m < NM; ++m) {
            const float x = v[1 + m + TG - 1 - t];
            const u64 vv = pack2(x, x);
#pragma unroll
            for (int h = 0; h < DH; ++h) ffma2(acc[r][m * DH + h], vv, w[t][h]);
          }
      }
    }
  }
}

template <int NC>
__device__ __forceinline__ void gemm_lowrate(const float* __restrict__ Rs, const float* __restrict__ Ys,
                                             float (&tmp)[4][5], int ty, int tx)
{
#pragma unroll 8
  for (int ll = 0; ll < RC_KC; ++ll) {
    const float4 a = *reinterpret_cast<const float4*>(Rs + ll * RC_RS + 4 * ty);
#pragma unroll
    for (int cc = 0; cc < NC; ++cc) {
      const float b = Ys[ll * RC_YS + tx + 16 * cc];
      tmp[0][cc] = fmaf(a.x, b, tmp[0][cc]); tmp[1][cc] = fmaf(a.y, b, tmp[1][cc]);
      tmp[2][cc] = fmaf(a.z, b, tmp[2][cc]); tmp[3][cc] = fmaf(a.w, b, tmp[3][cc]);
    }
  }
}

template <bool Y16>
__global__ void __launch_bounds__(256)
recon_f32_kernel(const SliceParams* __restrict__ sp, const BinParams* __restrict__ bp,
                 const float* const* __restrict__ upw, Peak* __restrict__ partials, int tiles_cap,
                 int max_templates, int c, long long k_a, Capture cap)
{
  const int bd = blockIdx.z;
  const BinParams B = bp[bd];
  const int row0 = blockIdx.y * RC_RT;
  if (row0 >= 2 * B.n_templates) return;
  const int g = blockIdx.x;
  const int kap0 = g * RC_CT;

  extern __shared__ __align__(16) float smem_r[];
  float* Rs = smem_r;                               // [RC_KC][RC_RS]
  float* Ys = Rs + RC_KC * RC_RS;                   // [RC_KC][RC_YS]
  float* rho = Ys + RC_KC * RC_YS;                  // [RC_RT][RC_RHO_S]
  float* wsm = rho + RC_RT * RC_RHO_S;              // [16][32]

  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  float acc[4][8];
#pragma unroll
  for (int r = 0; r < 4; ++r)
#pragma unroll
    for (int cc = 0; cc < 8; ++cc) acc[r][cc] = 0.f;

  for (int s = 0; s < B.n_slices; ++s) {
    const SliceParams P = sp[B.first_slice + s];
    const int d = P.d;
    const int Ks = (d == 1) ? RC_CT : (RC_CT >> P.log2d) + 2 * kKUp;
    const int r0 = (d == 1) ? kap0 : (kap0 >> P.log2d);
    const float* __restrict__ R = P.R32;
    const float* __restrict__ Y = reinterpret_cast<const float*>(P.Y);
    const int Lp = P.L_pad;
    float tmp[4][5];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int cc = 0; cc < 5; ++cc) tmp[r][cc] = 0.f;

    for (int l0 = 0; l0 < Lp; l0 += RC_KC) {
      __syncthreads();                               // also: previous slice's upsample has finished
      if (d > 1 && l0 == 0) {                        // stage this slice's interpolation weights
        const float* __restrict__ w = upw[P.log2d];  // [16][d]
        for (int e = tid; e < 16 * d; e += 256) wsm[(e / d) * 32 + (e % d)] = __ldg(w + e);
      }
#pragma unroll
      for (int i = 0; i < (RC_RT * RC_KC) / 256; ++i) {
        const int e = tid + 256 * i;
        const int ll = e % RC_KC, row = e / RC_KC;
        if (Y16) {                                   // packed fp16: R16[i / 128][l / 8][r16_lane(i % 128)][l % 8]
          const int i = row0 + row, l = l0 + ll;
          Rs[ll * RC_RS + row] = __half2float(P.R16[(((size_t)(i >> 7) * (Lp >> 3) + (l >> 3)) * 128 + r16_lane(i & 127)) * 8 + (l & 7)]);
        } else {
          Rs[ll * RC_RS + row] = __ldg(R + (size_t)(row0 + row) * Lp + l0 + ll);
        }
      }
      if (Y16) {                                     // packed fp16: Y16[row / 64][l / 8][row % 64][l % 8]
        const __half* __restrict__ Yh = reinterpret_cast<const __half*>(P.Y);
        for (int e = tid; e < Ks * RC_KC; e += 256) {
          const int le = e & 7, col = (e >> 3) % Ks, lg = (e >> 3) / Ks;
          const int r = r0 + col, l = l0 + lg * 8 + le;
          Ys[(lg * 8 + le) * RC_YS + col] =
              (r < P.y_rows_cap) ? __half2float(Yh[(size_t)(r >> 6) * (P.y_step64 >> 1) + ((size_t)(l >> 3) * 64 + (r & 63)) * 8 + le]) : 0.f;
        }
      } else {
        for (int e = tid; e < Ks * RC_KC; e += 256) {
          const int ll = e % RC_KC, col = e / RC_KC;
          const int r = r0 + col;
          Ys[ll * RC_YS + col] = (r < P.y_rows_cap) ? Y[(size_t)r * Lp + l0 + ll] : 0.f;
        }
      }
      __syncthreads();
      if (d == 1) {
#pragma unroll 8
        for (int ll = 0; ll < RC_KC; ++ll) {
          const float4 a = *reinterpret_cast<const float4*>(Rs + ll * RC_RS + 4 * ty);
          const float4 b0 = *reinterpret_cast<const float4*>(Ys + ll * RC_YS + 8 * tx);
          const float4 b1 = *reinterpret_cast<const float4*>(Ys + ll * RC_YS + 8 * tx + 4);
          const float av[4] = {a.x, a.y, a.z, a.w};
          const float bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
          for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int cc = 0; cc < 8; ++cc) acc[r][cc] = fmaf(av[r], bv[cc], acc[r][cc]);
        }
      } else if (d == 2) gemm_lowrate<5>(Rs, Ys, tmp, ty, tx);
      else if (d == 4) gemm_lowrate<3>(Rs, Ys, tmp, ty, tx);
      else gemm_lowrate<2>(Rs, Ys, tmp, ty, tx);
    }
    if (d > 1) {
      const int NC = (d == 2) ? 5 : (d == 4) ? 3 : 2;
      __syncthreads();                               // previous slice's readers of rho are done
      for (int cc = 0; cc < NC; ++cc) {
        const int col = tx + 16 * cc;
        if (col < Ks) {
#pragma unroll
          for (int r = 0; r < 4; ++r) rho[(4 * ty + r) * RC_RHO_S + col] = tmp[r][cc];
        }
      }
      __syncthreads();
      switch (d) {
        case 2: upsample_acc<2, 4>(acc, rho, wsm, ty, tx); break;
        case 4: upsample_acc<4, 4>(acc, rho, wsm, ty, tx); break;
        case 8: upsample_acc<8, 4>(acc, rho, wsm, ty, tx); break;
        case 16: upsample_acc<16, 4>(acc, rho, wsm, ty, tx); break;
        default: upsample_acc<32, 4>(acc, rho, wsm, ty, tx); break;
      }
    }
  }

  // ---- epilogue: |rho|^2, first maximum over the tile's valid columns, one Peak per template
  const int valid = min(RC_CT, c - kap0);           // ragged last tile of a chunk
#pragma unroll
  for (int t = 0; t < 2; ++t) {
    float bq = -1.f, bre = 0.f, bim = 0.f;
    int bk = 0x7fffffff;
#pragma unroll
    for (int cc = 0; cc < 8; ++cc) {
      const int kl = 8 * tx + cc;
      const float re = acc[2 * t][cc], im = acc[2 * t + 1][cc];
      const float q = re * re + im * im;
      if (kl < valid && q > bq) { bq = q; bre = re; bim = im; bk = kap0 + kl; }
    }
#pragma unroll
    for (int off = 8; off >= 1; off >>= 1) {
      const float oq = __shfl_xor_sync(0xffffffffu, bq, off);
      const float ore = __shfl_xor_sync(0xffffffffu, bre, off);
      const float oim = __shfl_xor_sync(0xffffffffu, bim, off);
      const int ok = __shfl_xor_sync(0xffffffffu, bk, off);
      if (oq > bq || (oq == bq && ok < bk)) { bq = oq; bre = ore; bim = oim; bk = ok; }
    }
    const int p = (row0 + 4 * ty) / 2 + t;
    if (tx == 0 && p < B.n_templates) {
      Peak pk; pk.q = bq; pk.kappa = bk; pk.re = bre; pk.im = bim;
      partials[((size_t)bd * tiles_cap + g) * max_templates + p] = pk;
    }
  }

  if (cap.snr != nullptr && cap.bd == bd) {         // test-only dense dump from the same accumulators
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int row = row0 + 4 * ty + r;
      if (row >= cap.rows) continue;
#pragma unroll
      for (int cc = 0; cc < 8; ++cc) {
        const int kl = 8 * tx + cc;
        const long long k = k_a + kap0 + kl;
        if (kl < valid && k >= cap.k_begin && k < cap.k_begin + cap.n)
          cap.snr[(size_t)row * cap.n + (k - cap.k_begin)] = acc[r][cc];
      }
    }
  }
}

void launch_recon_f32(const SliceParams* sp_dev, const BinParams* bp_dev, const BinParams* bp_host,
                      int n_bd, int max_rows_pad, const float* const* upw_dev, Peak* partials,
                      int tiles_cap, int max_templates, int c, int64_t k_a, Capture cap, bool packed16,
                      cudaStream_t st, int64_t* launches)
{
  (void)bp_host;
  const size_t smem = sizeof(float) * (RC_KC * RC_RS + RC_KC * RC_YS + RC_RT * RC_RHO_S + 16 * 32);
  const int n_tiles = (c + RC_CT - 1) / RC_CT;
  dim3 grid(n_tiles, (max_rows_pad + RC_RT - 1) / RC_RT, n_bd);
  if (packed16)
    recon_f32_kernel<true><<<grid, 256, smem, st>>>(sp_dev, bp_dev, upw_dev, partials, tiles_cap, max_templates,
                                                   c, (long long)k_a, cap);
  else
    recon_f32_kernel<false><<<grid, 256, smem, st>>>(sp_dev, bp_dev, upw_dev, partials, tiles_cap, max_templates,
                                                    c, (long long)k_a, cap);
  ++*launches;
}

// ------------------------------------------------------------------------------------------------
// A3 at the low rates, once per chunk:  Q[i, r] = sum_{slices s of the group} sum_l R^s[i, l] Y^s[r, l]
// (Y row r <-> low-rate index r - K_up, lloid_internal.h).  Plain register-tiled SGEMM "NT": CTA tile 128 rows x 128
// low-rate columns, 256 threads, 8 x 8 per thread, K chunks of 16 staged transposed in shared memory.  The fused
// f0 kernel used to recompute these products for every 128-sample tile with its 2 K_up halo (8x redundant at d = 32).
// ------------------------------------------------------------------------------------------------
constexpr int LG_T = 128, LG_K = 16, LG_S = LG_T + 4;

template <bool PK>
__global__ void __launch_bounds__(256, 2)
lowrate_gemm_f32_kernel(const SliceParams* __restrict__ sp, const Q32Group* __restrict__ groups, int c)
{
  const Q32Group G = groups[blockIdx.z];
  if (G.n_slices == 0) return;
  const int cols_needed = (c >> G.log2d) + 2 * kKUp;
  const int j0 = blockIdx.x * LG_T, row0 = blockIdx.y * LG_T;
  if (j0 >= cols_needed || row0 >= G.rows_pad) return;

  __shared__ __align__(16) float As[LG_K][LG_S], Bs[LG_K][LG_S];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  // this thread stages row lr, k = lk .. lk + 7 of both tiles (a lane pair reads 64 contiguous bytes); the upper k half
  // is stored with the row index XOR 16, so a warp's transposed stores fall into 32 different banks
  const int lr = tid >> 1, lk = (tid & 1) * 8, lc = lr ^ ((tid & 1) * 16);
  u64 acc[8][4];                                        // [row][column pair], packed fp32 x 2
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0ull;

  for (int s = 0; s < G.n_slices; ++s) {
    const SliceParams P = sp[G.slice[s]];
    const bool y_ok = j0 + lr < P.y_rows_cap;
    float4 a0, a1, b0 = make_float4(0.f, 0.f, 0.f, 0.f), b1 = b0;
    int r_step, y_step;
    const char* Rb = base8_R<PK>(P, row0 + lr, lk, r_step);
    const char* Yb = base8_Y<PK>(P, j0 + lr, lk, y_step);
    load8<PK, true>(Rb, a0, a1);
    if (y_ok) load8<PK, false>(Yb, b0, b1);
    for (int l0 = 0; l0 < P.L_pad; l0 += LG_K) {
      __syncthreads();
      As[lk + 0][lc] = a0.x; As[lk + 1][lc] = a0.y; As[lk + 2][lc] = a0.z; As[lk + 3][lc] = a0.w;
      As[lk + 4][lc] = a1.x; As[lk + 5][lc] = a1.y; As[lk + 6][lc] = a1.z; As[lk + 7][lc] = a1.w;
      Bs[lk + 0][lc] = b0.x; Bs[lk + 1][lc] = b0.y; Bs[lk + 2][lc] = b0.z; Bs[lk + 3][lc] = b0.w;
      Bs[lk + 4][lc] = b1.x; Bs[lk + 5][lc] = b1.y; Bs[lk + 6][lc] = b1.z; Bs[lk + 7][lc] = b1.w;
      __syncthreads();
      if (l0 + LG_K < P.L_pad) {                     // next chunk, in flight during the multiply
        Rb += (LG_K / 8) * r_step; Yb += (LG_K / 8) * y_step;
        load8<PK, true>(Rb, a0, a1);
        if (y_ok) load8<PK, false>(Yb, b0, b1);
      }
#pragma unroll
      for (int k = 0; k < LG_K; ++k) {
        // thread tile: rows 8 ty + i, columns 4 tx + j and 64 + 4 tx + j (16 B lane stride: no bank conflicts)
        const int sw = (k >> 3) * 16;
        const float4 av0 = *reinterpret_cast<const float4*>(&As[k][(ty * 8) ^ sw]), av1 = *reinterpret_cast<const float4*>(&As[k][(ty * 8 + 4) ^ sw]);
        const float4 bv0 = *reinterpret_cast<const float4*>(&Bs[k][(tx * 4) ^ sw]), bv1 = *reinterpret_cast<const float4*>(&Bs[k][(64 + tx * 4) ^ sw]);
        const float a[8] = {av0.x, av0.y, av0.z, av0.w, av1.x, av1.y, av1.z, av1.w};
        const u64 b[4] = {pack2(bv0.x, bv0.y), pack2(bv0.z, bv0.w), pack2(bv1.x, bv1.y), pack2(bv1.z, bv1.w)};
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const u64 aa = pack2(a[i], a[i]);
#pragma unroll
          for (int j = 0; j < 4; ++j) ffma2(acc[i][j], aa, b[j]);
        }
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    float* q = G.Q + (size_t)(row0 + ty * 8 + i) * G.q_cols + j0 + tx * 4;
    float4 o0, o1;
    unpack2(acc[i][0], o0.x, o0.y); unpack2(acc[i][1], o0.z, o0.w);
    unpack2(acc[i][2], o1.x, o1.y); unpack2(acc[i][3], o1.z, o1.w);
    *reinterpret_cast<float4*>(q) = o0;
    *reinterpret_cast<float4*>(q + 64) = o1;
  }
}

void launch_lowrate_gemm_f32(const SliceParams* sp_dev, const Q32Group* groups_dev, const Q32Group* groups_host, int n_groups,
                             int max_rows_pad, int c, bool packed16, cudaStream_t st, int64_t* launches)
{
  int max_cols = 0;
  for (int g = 0; g < n_groups; ++g)
    if (groups_host[g].n_slices) max_cols = std::max(max_cols, (c >> groups_host[g].log2d) + 2 * kKUp);
  if (max_cols == 0) return;
  dim3 grid((max_cols + LG_T - 1) / LG_T, (max_rows_pad + LG_T - 1) / LG_T, n_groups);
  if (packed16) lowrate_gemm_f32_kernel<true><<<grid, 256, 0, st>>>(sp_dev, groups_dev, c);
  else lowrate_gemm_f32_kernel<false><<<grid, 256, 0, st>>>(sp_dev, groups_dev, c);
  ++*launches;
}

// ------------------------------------------------------------------------------------------------
// fp32 path, second kernel: A3 of the d = 1 slices + A4 + A5 fused as in recon_f32_kernel, but the low-rate
// rho^(d) come precomputed from lowrate_gemm_f32_kernel: per rate the CTA stages a [128 rows x (128/d + 2 K_up)]
// window of Q and interpolates it into its register accumulators.
// CTA tile: 128 real rows (64 templates) x 128 f0 samples, 256 threads as 16 (row groups of 8) x 16 (column groups of
// 8), an 8 x 8 fp32 accumulator per thread.  K chunks of 16 are staged transposed (upper k half XOR-swizzled: no bank
// conflicts on the stores); the next chunk's global loads are in flight while the current one is multiplied.
// ------------------------------------------------------------------------------------------------
constexpr int RQ_T = 128, RQ_K = 16, RQ_S = RQ_T + 4, RQ_SB = 136;

// Window [RQ_T rows x (128/D + 2 K_up)] of rho^(d) -> shared memory.  The window starts on a multiple of 4 columns
// (r0 = 128 g / D), so it moves as float4; every thread has up to 8 loads in flight before its first store (with one
// load per loop trip the kernel spent 38 % of its stall samples on the store behind it).
template <int D>
__device__ __forceinline__ void stage_rho(float* __restrict__ rho, const float* __restrict__ Q, int qc, int q_left, int tid)
{
  constexpr int K4 = (RC_CT / D + 2 * kKUp) / 4;       // float4 per row
  constexpr int N4 = RQ_T * K4;
  constexpr int NIT = (N4 + 255) / 256;
#pragma unroll
  for (int i0 = 0; i0 < NIT; i0 += 8) {
    float4 v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      if (i0 + u >= NIT) continue;
      const int e = tid + 256 * (i0 + u);
      const int row = e / K4, c4 = (e % K4) * 4;
      v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (e < N4 && c4 < q_left) v[u] = __ldg(reinterpret_cast<const float4*>(Q + (size_t)row * qc + c4));
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      if (i0 + u >= NIT) continue;
      const int e = tid + 256 * (i0 + u);
      const int row = e / K4, c4 = (e % K4) * 4;
      if (e < N4) {
        const int col = (D >= 8) ? (c4 ^ (((row >> 3) & 1) * 16)) : c4;      // see upsample_acc2
        *reinterpret_cast<float4*>(rho + row * RQ_RHO_S + col) = v[u];
      }
    }
  }
}

template <bool PK>
__global__ void __launch_bounds__(256, 2)
recon_f32_q_kernel(const SliceParams* __restrict__ sp, const BinParams* __restrict__ bp,
                   const float* const* __restrict__ upw, const Q32Group* __restrict__ groups,
                   Peak* __restrict__ partials, int tiles_cap, int max_templates, int c, long long k_a, Capture cap)
{
  const int bd = blockIdx.z;
  if (groups[(size_t)bd * kNLowRates].rows_pad == 0) return;     // mixed fp16 bank: this bin is on the tensor kernels
  const BinParams B = bp[bd];
  const int row0 = blockIdx.y * RQ_T;
  if (row0 >= 2 * B.n_templates) return;
  const int g = blockIdx.x;
  const int kap0 = g * RC_CT;

  extern __shared__ __align__(16) float smem_r[];
  float* As = smem_r;                               // [RQ_K][RQ_S]  R tile, transposed
  // y tile, transposed and column-permuted: column c sits at 4 (c / 8) + c % 4 (+ 72 if c % 8 >= 4), so the 8 columns
  // of a thread are two float4 with a 16-byte lane stride (the plain layout's 32-byte stride is a 2-way conflict)
  float* Bs = As + RQ_K * RQ_S;                     // [RQ_K][RQ_SB]
  float* rho = Bs + RQ_K * RQ_SB;                   // [RQ_T][RQ_RHO_S]
  float* wsm = rho + RQ_T * RQ_RHO_S;               // [16][32]

  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int lr = tid >> 1, lk = (tid & 1) * 8, lc = lr ^ ((tid & 1) * 16);   // staging: row lr, k = lk .. lk + 7 (upper half swizzled)
  const int lcb = ((((lr >> 3) << 2) | (lr & 3)) ^ ((tid & 1) * 16)) + ((lr & 4) ? 72 : 0);
  u64 acc2[8][4];                                   // [row][column pair], packed fp32 x 2
#pragma unroll
  for (int r = 0; r < 8; ++r)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc2[r][j] = 0ull;

  // ---- d = 1 slices: K-chunked SGEMM straight into the accumulators
  for (int s = 0; s < B.n_slices; ++s) {
    const SliceParams P = sp[B.first_slice + s];
    if (P.d != 1) continue;
    const int Lp = P.L_pad;
    const bool y_ok = kap0 + lr < P.y_rows_cap;
    float4 a0, a1, b0 = make_float4(0.f, 0.f, 0.f, 0.f), b1 = b0;
    int r_step, y_step;
    const char* Rb = base8_R<PK>(P, row0 + lr, lk, r_step);
    const char* Yb = base8_Y<PK>(P, kap0 + lr, lk, y_step);
    load8<PK, true>(Rb, a0, a1);
    if (y_ok) load8<PK, false>(Yb, b0, b1);
    for (int l0 = 0; l0 < Lp; l0 += RQ_K) {
      __syncthreads();
      As[(lk + 0) * RQ_S + lc] = a0.x; As[(lk + 1) * RQ_S + lc] = a0.y; As[(lk + 2) * RQ_S + lc] = a0.z; As[(lk + 3) * RQ_S + lc] = a0.w;
      As[(lk + 4) * RQ_S + lc] = a1.x; As[(lk + 5) * RQ_S + lc] = a1.y; As[(lk + 6) * RQ_S + lc] = a1.z; As[(lk + 7) * RQ_S + lc] = a1.w;
      Bs[(lk + 0) * RQ_SB + lcb] = b0.x; Bs[(lk + 1) * RQ_SB + lcb] = b0.y; Bs[(lk + 2) * RQ_SB + lcb] = b0.z; Bs[(lk + 3) * RQ_SB + lcb] = b0.w;
      Bs[(lk + 4) * RQ_SB + lcb] = b1.x; Bs[(lk + 5) * RQ_SB + lcb] = b1.y; Bs[(lk + 6) * RQ_SB + lcb] = b1.z; Bs[(lk + 7) * RQ_SB + lcb] = b1.w;
      __syncthreads();
      if (l0 + RQ_K < Lp) {                          // next chunk, in flight during the multiply
        Rb += (RQ_K / 8) * r_step; Yb += (RQ_K / 8) * y_step;
        load8<PK, true>(Rb, a0, a1);
        if (y_ok) load8<PK, false>(Yb, b0, b1);
      }
#pragma unroll
      for (int k = 0; k < RQ_K; ++k) {
        const int sw = (k >> 3) * 16;
        const float4 av0 = *reinterpret_cast<const float4*>(As + k * RQ_S + ((ty * 8) ^ sw)), av1 = *reinterpret_cast<const float4*>(As + k * RQ_S + ((ty * 8 + 4) ^ sw));
        const float4 bv0 = *reinterpret_cast<const float4*>(Bs + k * RQ_SB + ((tx * 4) ^ sw)), bv1 = *reinterpret_cast<const float4*>(Bs + k * RQ_SB + 72 + ((tx * 4) ^ sw));
        const float a[8] = {av0.x, av0.y, av0.z, av0.w, av1.x, av1.y, av1.z, av1.w};
        const u64 b[4] = {pack2(bv0.x, bv0.y), pack2(bv0.z, bv0.w), pack2(bv1.x, bv1.y), pack2(bv1.z, bv1.w)};
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const u64 aa = pack2(a[i], a[i]);
#pragma unroll
          for (int j = 0; j < 4; ++j) ffma2(acc2[i][j], aa, b[j]);
        }
      }
    }
  }

  // ---- low rates: window of the precomputed rho^(d), interpolated (A4)
  for (int l2 = 1; l2 < kMaxRates; ++l2) {
    const Q32Group* G = groups + (size_t)bd * kNLowRates + (l2 - 1);
    if (G->n_slices == 0) continue;
    const int d = 1 << l2;
    const int r0 = kap0 >> l2;
    const float* __restrict__ Q = G->Q + (size_t)row0 * G->q_cols + r0;
    const int qc = G->q_cols, q_left = G->q_cols - r0;
    __syncthreads();                                 // previous readers of rho / wsm are done
    {
      const float* __restrict__ w = upw[l2];         // [16][d]
      for (int e = tid; e < 16 * d; e += 256) wsm[(e / d) * 32 + (e % d)] = __ldg(w + e);
    }
    switch (d) {
      case 2: stage_rho<2>(rho, Q, qc, q_left, tid); __syncthreads(); upsample_acc2<2>(acc2, rho, wsm, ty, tx); break;
      case 4: stage_rho<4>(rho, Q, qc, q_left, tid); __syncthreads(); upsample_acc2<4>(acc2, rho, wsm, ty, tx); break;
      case 8: stage_rho<8>(rho, Q, qc, q_left, tid); __syncthreads(); upsample_acc2<8>(acc2, rho, wsm, ty, tx); break;
      case 16: stage_rho<16>(rho, Q, qc, q_left, tid); __syncthreads(); upsample_acc2<16>(acc2, rho, wsm, ty, tx); break;
      default: stage_rho<32>(rho, Q, qc, q_left, tid); __syncthreads(); upsample_acc2<32>(acc2, rho, wsm, ty, tx); break;
    }
  }

  // ---- epilogue: |rho|^2, first maximum over the tile's valid columns, one Peak per template
  float acc[8][8];
#pragma unroll
  for (int r = 0; r < 8; ++r)
#pragma unroll
    for (int j = 0; j < 4; ++j) unpack2(acc2[r][j], acc[r][2 * j], acc[r][2 * j + 1]);
  const int valid = min(RC_CT, c - kap0);           // ragged last tile of a chunk
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    float bq = -1.f, bre = 0.f, bim = 0.f;
    int bk = 0x7fffffff;
#pragma unroll
    for (int cc = 0; cc < 8; ++cc) {
      const int kl = 8 * tx + cc;
      const float re = acc[2 * t][cc], im = acc[2 * t + 1][cc];
      const float q = re * re + im * im;
      if (kl < valid && q > bq) { bq = q; bre = re; bim = im; bk = kap0 + kl; }
    }
#pragma unroll
    for (int off = 8; off >= 1; off >>= 1) {
      const float oq = __shfl_xor_sync(0xffffffffu, bq, off);
      const float ore = __shfl_xor_sync(0xffffffffu, bre, off);
      const float oim = __shfl_xor_sync(0xffffffffu, bim, off);
      const int ok = __shfl_xor_sync(0xffffffffu, bk, off);
      if (oq > bq || (oq == bq && ok < bk)) { bq = oq; bre = ore; bim = oim; bk = ok; }
    }
    const int p = (row0 + 8 * ty) / 2 + t;
    if (tx == 0 && p < B.n_templates) {
      Peak pk; pk.q = bq; pk.kappa = bk; pk.re = bre; pk.im = bim;
      partials[((size_t)bd * tiles_cap + g) * max_templates + p] = pk;
    }
  }

  if (cap.snr != nullptr && cap.bd == bd) {         // test-only dense dump from the same accumulators
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      const int row = row0 + 8 * ty + r;
      if (row >= cap.rows) continue;
#pragma unroll
      for (int cc = 0; cc < 8; ++cc) {
        const int kl = 8 * tx + cc;
        const long long k = k_a + kap0 + kl;
        if (kl < valid && k >= cap.k_begin && k < cap.k_begin + cap.n)
          cap.snr[(size_t)row * cap.n + (k - cap.k_begin)] = acc[r][cc];
      }
    }
  }
}

void launch_recon_f32_q(const SliceParams* sp_dev, const BinParams* bp_dev, int n_bd, int max_rows_pad,
                        const float* const* upw_dev, const Q32Group* groups_dev, Peak* partials, int tiles_cap,
                        int max_templates, int c, int64_t k_a, Capture cap, bool packed16, cudaStream_t st, int64_t* launches)
{
  const size_t smem = sizeof(float) * (RQ_K * RQ_S + RQ_K * RQ_SB + RQ_T * RQ_RHO_S + 16 * 32);
  const int n_tiles = (c + RC_CT - 1) / RC_CT;
  dim3 grid(n_tiles, (max_rows_pad + RQ_T - 1) / RQ_T, n_bd);
  if (packed16)
    recon_f32_q_kernel<true><<<grid, 256, smem, st>>>(sp_dev, bp_dev, upw_dev, groups_dev, partials, tiles_cap, max_templates,
                                                     c, (long long)k_a, cap);
  else
    recon_f32_q_kernel<false><<<grid, 256, smem, st>>>(sp_dev, bp_dev, upw_dev, groups_dev, partials, tiles_cap, max_templates,
                                                      c, (long long)k_a, cap);
  ++*launches;
}

// Opt-in shared memory is a per-device, per-function attribute: set once per bank at finalize (after cudaSetDevice),
// always to the architecture maximum, so banks on several devices or of different sizes never interfere.
int configure_f32_kernels()
{
  const int m = 227 * 1024;
  cudaError_t e = set_max_dyn_smem(fir_f32_kernel);
  if (e == cudaSuccess) e = set_max_dyn_smem(recon_f32_kernel<false>);
  if (e == cudaSuccess) e = set_max_dyn_smem(recon_f32_kernel<true>);
  if (e == cudaSuccess) e = set_max_dyn_smem(recon_f32_q_kernel<false>);
  if (e == cudaSuccess) e = set_max_dyn_smem(recon_f32_q_kernel<true>);
  return e == cudaSuccess ? 0 : 1;
}

}  // namespace lloid
