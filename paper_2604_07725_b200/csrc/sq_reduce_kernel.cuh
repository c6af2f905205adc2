// sq_reduce_kernel.cuh -- kernel 2 (step a7): per-sequence varlen reductions over cu_seqlens.
//
//   seq_mean_logprob  = mean target_logprob over valid targets
//   seq_mean_entropy  = mean entropy
//   seq_mean_conf     = C(tau) = (1/|tau|) sum_i c(i)                       (Eq. 4)
//   seq_min_window_conf = min_j (1/w') sum_{i=j}^{j+w'-1} c(i),  w' = min(w, L), stride 1
//
// HBM-bound (12 B/token).  Three launches:
//   tile_scan : exclusive scan of ceil(L_b / TILE) -> tile_base[B+1]           (1 CTA)
//   tile_part : one CTA per (sequence, tile of TILE = 8192 tokens): coalesced partial sums and the minimum
//               window sum among the windows that START in the tile.  The window sums are
//               S(j) = S(j0) + sum_{i=j0+1..j} (c[i+w'-1] - c[i-1]): S(j0) is summed directly and the
//               differences are scanned per warp, so fp32 error does not grow with the sequence.
//   seq_final : one warp per sequence folds its tiles' partials in fixed order (fp64 accumulators).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace sq {

#ifndef SQ_RED_TILE
#define SQ_RED_TILE 8192
#endif
#ifndef SQ_RED_UNROLL
#define SQ_RED_UNROLL 8
#endif
constexpr int RED_TILE = SQ_RED_TILE;   // tokens per CTA
constexpr int RED_UNROLL = SQ_RED_UNROLL;   // independent loads per array in flight per thread
constexpr int RED_THREADS = 256;
constexpr int RED_WARPS = RED_THREADS / 32;
constexpr int RED_PER_WARP = RED_TILE / RED_WARPS;   // 512 window starts per warp

struct ReduceParams {
  long long T;
  int B, V, window;
  const float* lp;
  const float* ent;
  const float* conf;
  const int32_t* targets;     // may be null: all valid
  const int32_t* cu;
  int* tile_base;             // [B+1]
  int* tile_seq;              // [tiles] sequence that owns each tile (written by tile_scan)
  float4* part_sum;           // [tiles] (sum_lp, n_valid, sum_ent, sum_conf)
  float* part_min;            // [tiles] min window SUM among windows starting in the tile (+inf if none)
  float* out_lp; float* out_ent; float* out_conf; float* out_min;
};

__global__ void __launch_bounds__(1024) sq_reduce_tile_scan_kernel(const ReduceParams p) {
  __shared__ int warp_tot[32];
  __shared__ int carry_s;
  if (threadIdx.x == 0) { carry_s = 0; p.tile_base[0] = 0; }
  __syncthreads();
  for (int b0 = 0; b0 < p.B; b0 += 1024) {
    const int b = b0 + threadIdx.x;
    int n = 0;
    if (b < p.B) {
      const int L = p.cu[b + 1] - p.cu[b];
      n = L > 0 ? (L + RED_TILE - 1) / RED_TILE : 0;
    }
    int x = n;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, x, off);
      if ((threadIdx.x & 31) >= off) x += y;
    }
    if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x < 32) {
      int t = warp_tot[threadIdx.x];
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, t, off);
        if (threadIdx.x >= off) t += y;
      }
      warp_tot[threadIdx.x] = t;
    }
    __syncthreads();
    const int wbase = (threadIdx.x >> 5) ? warp_tot[(threadIdx.x >> 5) - 1] : 0;
    const int incl = carry_s + wbase + x;
    if (b < p.B) {
      p.tile_base[b + 1] = incl;
      for (int i = incl - n; i < incl; ++i) p.tile_seq[i] = b;   // n = ceil(L / 4096): a handful per sequence
    }
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = incl;
    __syncthreads();
  }
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

__global__ void __launch_bounds__(RED_THREADS) sq_reduce_tile_part_kernel(const ReduceParams p) {
  __shared__ float sh[RED_WARPS][7];
  const int tile = blockIdx.x;
  const int total_tiles = p.tile_base[p.B];
  if (tile >= total_tiles) return;
  const int b = p.tile_seq[tile];
  const long long seq0 = p.cu[b];
  const int L = p.cu[b + 1] - p.cu[b];
  const int t_in = (tile - p.tile_base[b]) * RED_TILE;       // first token of the tile, in the sequence
  const int n_tok = min(RED_TILE, L - t_in);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- partial sums over the tile's tokens (coalesced; 4 independent loads per array in flight)
  float a_lp = 0.f, a_n = 0.f, a_en = 0.f, a_cf = 0.f;
  {
    const long long t0 = seq0 + t_in;
    const float* lp = p.lp + t0; const float* en = p.ent + t0; const float* cf = p.conf + t0;
    const int32_t* tg = p.targets ? p.targets + t0 : nullptr;
    for (int i0 = 0; i0 < n_tok; i0 += RED_UNROLL * RED_THREADS) {
      float vl[RED_UNROLL], ve[RED_UNROLL], vc[RED_UNROLL]; int vt[RED_UNROLL];
#pragma unroll
      for (int q = 0; q < RED_UNROLL; ++q) {
        const int i = i0 + q * RED_THREADS + threadIdx.x;
        const bool in = i < n_tok;
        vl[q] = in ? __ldg(lp + i) : 0.f;
        ve[q] = in ? __ldg(en + i) : 0.f;
        vc[q] = in ? __ldg(cf + i) : 0.f;
        vt[q] = in ? (tg ? __ldg(tg + i) : 0) : -1;
      }
#pragma unroll
      for (int q = 0; q < RED_UNROLL; ++q) {
        const bool valid = (vt[q] >= 0) && (vt[q] < p.V || !tg);
        if (valid) { a_lp += vl[q]; a_n += 1.f; }
        a_en += ve[q];
        a_cf += vc[q];
      }
    }
  }

  // ---- sliding windows that start in this tile
  const int w = min(p.window, L);
  const int n_win = L - w + 1;
  const int j0 = t_in;
  const int j1 = min(t_in + RED_TILE, n_win);   // window starts [j0, j1)
  const float* c = p.conf + seq0;
  float a_s0 = 0.f;
  if (j0 < j1) {
    for (int i = threadIdx.x; i < w; i += RED_THREADS) a_s0 += c[j0 + i];   // S(j0), summed directly
  }
  a_lp = warp_sum(a_lp); a_n = warp_sum(a_n); a_en = warp_sum(a_en); a_cf = warp_sum(a_cf); a_s0 = warp_sum(a_s0);

  // each warp scans the differences of its 512 consecutive window starts
  float run = 0.f;                 // S(j) - S(first start of this warp's strip), inclusive
  float wmin = CUDART_INF_F;       // min over the strip of that relative sum
  const int s_begin = j0 + warp * RED_PER_WARP;
  float dl[RED_PER_WARP / 32];
#pragma unroll
  for (int r = 0; r < RED_PER_WARP / 32; ++r) {   // all difference loads first: 32 loads in flight per thread
    const int j = s_begin + r * 32 + lane;
    // strip-relative: the first start of the strip contributes 0; later starts add c[j+w-1] - c[j-1]
    const bool ld = (j < j1) && (j > s_begin);
    const float a = ld ? __ldg(c + j + w - 1) : 0.f;
    const float bq = ld ? __ldg(c + j - 1) : 0.f;
    dl[r] = a - bq;
  }
#pragma unroll
  for (int r = 0; r < RED_PER_WARP / 32; ++r) {
    const int j = s_begin + r * 32 + lane;
    const bool in = (j < j1);
    float x = dl[r];
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const float y = __shfl_up_sync(0xffffffffu, x, off);
      if (lane >= off) x += y;
    }
    x += run;
    if (in) wmin = fminf(wmin, x);
    run = __shfl_sync(0xffffffffu, x, 31);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) wmin = fminf(wmin, __shfl_xor_sync(0xffffffffu, wmin, off));
  // the strip's total, plus the step from its last start to the next strip's first start
  float step = 0.f;
  {
    const int jn = s_begin + RED_PER_WARP;   // first start of the next strip
    if (jn < j1) step = c[jn + w - 1] - c[jn - 1];
  }
  if (lane == 0) {
    sh[warp][0] = a_lp; sh[warp][1] = a_n; sh[warp][2] = a_en; sh[warp][3] = a_cf;
    sh[warp][4] = wmin; sh[warp][5] = run + step; sh[warp][6] = a_s0;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    float s_lp = 0.f, s_n = 0.f, s_en = 0.f, s_cf = 0.f;
    float base = 0.f, best = CUDART_INF_F;
    for (int q = 0; q < RED_WARPS; ++q) base += sh[q][6];   // S(j0), fixed order
    for (int q = 0; q < RED_WARPS; ++q) {
      s_lp += sh[q][0]; s_n += sh[q][1]; s_en += sh[q][2]; s_cf += sh[q][3];
      best = fminf(best, base + sh[q][4]);   // +inf stays +inf for strips without windows
      base += sh[q][5];
    }
    p.part_sum[tile] = make_float4(s_lp, s_n, s_en, s_cf);
    p.part_min[tile] = best;
  }
}

__global__ void __launch_bounds__(128) sq_reduce_seq_final_kernel(const ReduceParams p) {
  const int b = blockIdx.x * 4 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (b >= p.B) return;
  const int L = p.cu[b + 1] - p.cu[b];
  const int t0 = p.tile_base[b], t1 = p.tile_base[b + 1];
  double s_lp = 0.0, s_n = 0.0, s_en = 0.0, s_cf = 0.0;
  float best = CUDART_INF_F;
  for (int t = t0 + lane; t < t1; t += 32) {
    const float4 v = p.part_sum[t];
    s_lp += v.x; s_n += v.y; s_en += v.z; s_cf += v.w;
    best = fminf(best, p.part_min[t]);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    s_lp += __shfl_xor_sync(0xffffffffu, s_lp, off);
    s_n += __shfl_xor_sync(0xffffffffu, s_n, off);
    s_en += __shfl_xor_sync(0xffffffffu, s_en, off);
    s_cf += __shfl_xor_sync(0xffffffffu, s_cf, off);
    best = fminf(best, __shfl_xor_sync(0xffffffffu, best, off));
  }
  if (lane == 0) {
    const float nan = CUDART_NAN_F;
    if (L <= 0) {
      p.out_lp[b] = nan; p.out_ent[b] = nan; p.out_conf[b] = nan; p.out_min[b] = nan;
    } else {
      const int w = min(p.window, L);
      p.out_lp[b] = (s_n > 0.0) ? (float)(s_lp / s_n) : nan;
      p.out_ent[b] = (float)(s_en / (double)L);
      p.out_conf[b] = (float)(s_cf / (double)L);
      p.out_min[b] = best / (float)w;
    }
  }
}

}  // namespace sq
