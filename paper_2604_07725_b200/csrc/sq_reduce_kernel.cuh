// sq_reduce_kernel.cuh -- kernel 2 (step a7): per-sequence varlen reductions over cu_seqlens.
//
//   seq_mean_logprob  = mean target_logprob over valid targets
//   seq_mean_entropy  = mean entropy
//   seq_mean_conf     = C(tau) = (1/|tau|) sum_i c(i)                       (Eq. 4)
//   seq_min_window_conf = min_j (1/w') sum_{i=j}^{j+w'-1} c(i),  w' = min(w, L), stride 1
//
// HBM-bound (12 B/token).  Three launches, the 2nd and 3rd with programmatic stream serialization so that
// their launch latency overlaps the kernel before them:
//   tile_scan : exclusive scan of ceil(L_b / TILE) -> tile_base[B+1], tile -> sequence map, NaNs for
//               empty sequences                                                  (1 CTA)
//   tile_part : one CTA per (sequence, tile of TILE = 8192 tokens): coalesced partial sums and the minimum
//               window sum among the windows that START in the tile.  The window sums are
//               S(j) = S(j0) + sum_{i=j0+1..j} (c[i+w'-1] - c[i-1]): S(j0) is summed directly and the
//               differences are parked in shared memory and scanned (32 per thread + one block scan),
//               so fp32 error does not grow with the sequence.
//   seq_final : one warp per sequence folds its tiles' partials in fixed order (fp64 accumulators):
//               deterministic, no float atomics.  (Folding in the tile CTA that finishes last was
//               measured slower: the fence + atomic tail keeps every CTA's registers 2 us longer.)
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
constexpr int RED_SMEM_BYTES = (RED_TILE + RED_TILE / 32 + 32) * 4;   // padded difference array

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
  // thread t owns the `per` consecutive sequences [t*per, (t+1)*per): one block scan in total
  const int per = (p.B + 1023) / 1024;
  const int b_lo = threadIdx.x * per, b_hi = min(p.B, b_lo + per);
  int mine = 0;
  for (int b = b_lo; b < b_hi; ++b) {
    const int L = p.cu[b + 1] - p.cu[b];
    mine += L > 0 ? (L + RED_TILE - 1) / RED_TILE : 0;
  }
  int x = mine;
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
  int base = ((threadIdx.x >> 5) ? warp_tot[(threadIdx.x >> 5) - 1] : 0) + x - mine;   // exclusive prefix
  if (threadIdx.x == 0) p.tile_base[0] = 0;
  for (int b = b_lo; b < b_hi; ++b) {
    const int L = p.cu[b + 1] - p.cu[b];
    const int n = L > 0 ? (L + RED_TILE - 1) / RED_TILE : 0;
    for (int i = 0; i < n; ++i) p.tile_seq[base + i] = b;   // n = ceil(L / RED_TILE): a handful per sequence
    base += n;
    p.tile_base[b + 1] = base;
    if (n == 0) {   // empty sequence: no tile CTA will ever visit it
      const float nan = CUDART_NAN_F;
      p.out_lp[b] = nan; p.out_ent[b] = nan; p.out_conf[b] = nan; p.out_min[b] = nan;
    }
  }
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

// Partial sums of one tile: FULL = all RED_TILE tokens present (no bounds checks), HAS_TG = targets given.
template <bool FULL, bool HAS_TG>
__device__ __forceinline__ void tile_sums(const ReduceParams& p, long long t0, int n_tok, float& a_lp, float& a_n,
                                          float& a_en, float& a_cf) {
  const float* lp = p.lp + t0; const float* en = p.ent + t0; const float* cf = p.conf + t0;
  const int32_t* tg = HAS_TG ? p.targets + t0 : nullptr;
  for (int i0 = 0; i0 < (FULL ? RED_TILE : n_tok); i0 += RED_UNROLL * RED_THREADS) {
    float vl[RED_UNROLL], ve[RED_UNROLL], vc[RED_UNROLL]; int vt[RED_UNROLL];
#pragma unroll
    for (int q = 0; q < RED_UNROLL; ++q) {   // all loads of the batch first: 3-4 x RED_UNROLL in flight per thread
      const int i = i0 + q * RED_THREADS + threadIdx.x;
      const bool in = FULL || (i < n_tok);
      vl[q] = in ? __ldg(lp + i) : 0.f;
      ve[q] = in ? __ldg(en + i) : 0.f;
      vc[q] = in ? __ldg(cf + i) : 0.f;
      if (HAS_TG) vt[q] = in ? __ldg(tg + i) : -1; else vt[q] = in ? 0 : -1;
    }
#pragma unroll
    for (int q = 0; q < RED_UNROLL; ++q) {
      const bool valid = HAS_TG ? ((unsigned)vt[q] < (unsigned)p.V) : (vt[q] >= 0);
      a_lp += valid ? vl[q] : 0.f;
      a_n += valid ? 1.f : 0.f;
      a_en += ve[q];
      a_cf += vc[q];
    }
  }
}

__device__ __forceinline__ int red_pad(int i) { return i + (i >> 5); }   // conflict-free 32-float runs per thread

__global__ void __launch_bounds__(RED_THREADS) sq_reduce_tile_part_kernel(const ReduceParams p) {
  extern __shared__ float s_d[];                 // window-sum differences of the tile, padded
  __shared__ float sh[RED_WARPS][8];
  cudaGridDependencySynchronize();               // launched with programmatic serialization behind tile_scan
  const int tile = blockIdx.x;
  const int total_tiles = p.tile_base[p.B];
  if (tile >= total_tiles) return;
  const int b = p.tile_seq[tile];
  const long long seq0 = p.cu[b];
  const int L = p.cu[b + 1] - p.cu[b];
  const int t_in = (tile - p.tile_base[b]) * RED_TILE;       // first token of the tile, in the sequence
  const int n_tok = min(RED_TILE, L - t_in);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- partial sums over the tile's tokens (coalesced)
  float a_lp = 0.f, a_n = 0.f, a_en = 0.f, a_cf = 0.f;
  if (n_tok == RED_TILE) {
    if (p.targets) tile_sums<true, true>(p, seq0 + t_in, n_tok, a_lp, a_n, a_en, a_cf);
    else tile_sums<true, false>(p, seq0 + t_in, n_tok, a_lp, a_n, a_en, a_cf);
  } else {
    if (p.targets) tile_sums<false, true>(p, seq0 + t_in, n_tok, a_lp, a_n, a_en, a_cf);
    else tile_sums<false, false>(p, seq0 + t_in, n_tok, a_lp, a_n, a_en, a_cf);
  }

  // ---- sliding windows that start in this tile: S(j) = S(j0) + sum_{i=j0+1..j} (c[i+w-1] - c[i-1])
  const int w = min(p.window, L);
  const int n_win = L - w + 1;
  const int j0 = t_in;
  const int j1 = min(t_in + RED_TILE, n_win);   // window starts [j0, j1)
  const float* c = p.conf + seq0;
  float a_s0 = 0.f;
  if (j0 < j1) {
    for (int i = threadIdx.x; i < w; i += RED_THREADS) a_s0 += __ldg(c + j0 + i);   // S(j0), summed directly
    // differences, loaded coalesced and parked in shared memory (D[j0] = 0)
#pragma unroll 8
    for (int r = 0; r < RED_TILE / RED_THREADS; ++r) {
      const int i = r * RED_THREADS + threadIdx.x;
      const int j = j0 + i;
      float dlt = 0.f;
      if (j < j1 && i > 0) dlt = __ldg(c + j + w - 1) - __ldg(c + j - 1);
      s_d[red_pad(i)] = dlt;
    }
  }
  a_lp = warp_sum(a_lp); a_n = warp_sum(a_n); a_en = warp_sum(a_en); a_cf = warp_sum(a_cf); a_s0 = warp_sum(a_s0);
  __syncthreads();

  // each thread scans its 32 consecutive window starts, then one block scan of the 256 totals
  constexpr int PER_THREAD = RED_TILE / RED_THREADS;
  float run = 0.f, tmin = CUDART_INF_F;
  if (j0 < j1) {
    const int base = threadIdx.x * PER_THREAD;
#pragma unroll
    for (int i = 0; i < PER_THREAD; ++i) {
      run += s_d[red_pad(base + i)];
      if (j0 + base + i < j1) tmin = fminf(tmin, run);
    }
  }
  float incl = run;                               // inclusive scan of the thread totals
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const float y = __shfl_up_sync(0xffffffffu, incl, off);
    if (lane >= off) incl += y;
  }
  if (lane == 31) sh[warp][5] = incl;
  if (lane == 0) { sh[warp][0] = a_lp; sh[warp][1] = a_n; sh[warp][2] = a_en; sh[warp][3] = a_cf; sh[warp][6] = a_s0; }
  __syncthreads();
  float woff = 0.f;
  for (int q = 0; q < warp; ++q) woff += sh[q][5];
  float wmin = tmin + (woff + incl - run);        // +inf stays +inf for threads without a window
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) wmin = fminf(wmin, __shfl_xor_sync(0xffffffffu, wmin, off));
  if (lane == 0) sh[warp][4] = wmin;
  __syncthreads();
  if (threadIdx.x == 0) {
    float s_lp = 0.f, s_n = 0.f, s_en = 0.f, s_cf = 0.f, s0 = 0.f, best = CUDART_INF_F;
    for (int q = 0; q < RED_WARPS; ++q) {        // fixed order: deterministic
      s_lp += sh[q][0]; s_n += sh[q][1]; s_en += sh[q][2]; s_cf += sh[q][3]; s0 += sh[q][6];
      best = fminf(best, sh[q][4]);
    }
    p.part_sum[tile] = make_float4(s_lp, s_n, s_en, s_cf);
    p.part_min[tile] = s0 + best;
  }
}

__global__ void __launch_bounds__(128) sq_reduce_seq_final_kernel(const ReduceParams p) {
  cudaGridDependencySynchronize();               // launched with programmatic serialization behind tile_part
  const int b = blockIdx.x * 4 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (b >= p.B) return;
  const int L = p.cu[b + 1] - p.cu[b];
  if (L <= 0) return;                            // tile_scan already wrote the NaNs
  const int t0 = p.tile_base[b], t1 = p.tile_base[b + 1];
  double s_lp = 0.0, s_n = 0.0, s_en = 0.0, s_cf = 0.0;
  float best = CUDART_INF_F;
  for (int t = t0 + lane; t < t1; t += 32) {     // fixed order: deterministic
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
    const int w = min(p.window, L);
    p.out_lp[b] = (s_n > 0.0) ? (float)(s_lp / s_n) : CUDART_NAN_F;
    p.out_ent[b] = (float)(s_en / (double)L);
    p.out_conf[b] = (float)(s_cf / (double)L);
    p.out_min[b] = best / (float)w;
  }
}

}  // namespace sq
