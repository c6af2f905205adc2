// sq_reduce_kernel.cuh -- kernel 2 (step a7): per-sequence varlen reductions over cu_seqlens.
//
//   seq_mean_logprob  = mean target_logprob over valid targets
//   seq_mean_entropy  = mean entropy
//   seq_mean_conf     = C(tau) = (1/|tau|) sum_i c(i)                       (Eq. 4)
//   seq_min_window_conf = min_j (1/w') sum_{i=j}^{j+w'-1} c(i),  w' = min(w, L), stride 1
//
// HBM-bound (12 B/token).  Large inputs take three launches, each with programmatic stream serialization so that its
// launch latency overlaps the kernel before it; small ones (the scoring pipeline) a single launch that does the same
// work per tile (sq_reduce_fused_kernel, at the end of this file):
//   tile_scan : tile i of a sequence covers the block of TILE = 8192 tokens that starts at (s0 & ~3) + i*TILE of the
//               packed arrays (s0 = the sequence's first token), so every tile's 16-byte vectors are aligned and only
//               a sequence's last tile is ragged.  Exclusive scan of the tiles per sequence -> tile_base[B+1],
//               tile -> sequence map, NaNs for empty sequences                   (1 CTA)
//   tile_part : one CTA per tile: partial sums from 16-byte loads, and the minimum window sum among the windows
//               that START in the tile.  The window sums are S(j) = S(ja) + sum_{m=ja..j-1} (c[m+w'] - c[m]):
//               S(ja) for the tile's first token is summed directly; the differences are formed in registers
//               (c[m] is the vector just loaded for the sums, c[m+w'] two aligned vectors funnelled by w' mod 4),
//               parked in shared memory and scanned (32 per thread from 16-byte shared loads + one block scan),
//               so fp32 error does not grow with the sequence.  Rows of 1024 tokens are classified CTA-uniformly
//               (inside the difference range / inside the tile only / ragged); ragged rows take scalar loads.
//               Measured stand-alone (4096 sequences, 3.6e7 tokens): 0.101 ms for the three launches = 4.25 TB/s;
//               the same launches with the window work removed take 0.084 ms, so ~14 us of the total is launch
//               structure (scan + final + gaps) and ~17 us the look-ahead loads and the scan.
//   seq_final : one warp per sequence folds its tiles' partials in fixed order (fp64 accumulators):
//               deterministic, no float atomics.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace sq {

#ifndef SQ_RED_TILE
#define SQ_RED_TILE 8192
#endif
#ifndef SQ_RED_NB
#define SQ_RED_NB 2
#endif
constexpr int RED_TILE = SQ_RED_TILE;     // tokens per tile = per CTA
constexpr int RED_THREADS = 256;
constexpr int RED_WARPS = RED_THREADS / 32;
constexpr int RED_PER_THREAD = RED_TILE / RED_THREADS;            // 32 consecutive differences per thread
constexpr int RED_CHUNKS = RED_TILE / 4 / RED_THREADS;            // 16-byte vectors per thread and array: 8
constexpr int RED_SMEM_BYTES = (RED_TILE + RED_TILE / 8) * 4;     // 4 pad floats per 32: 16-byte shared loads stay conflict-free

struct ReduceParams {
  long long T;
  int B, V, window;
  int vec;                    // 1: lp / ent / conf / targets are 16-byte aligned (vector loads); 0: scalar loads
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
  int* seq_done;              // [B] tiles of each sequence finished so far (single-launch form; all zero between runs)
};

// tiles of the sequence [s0, s1): blocks of RED_TILE tokens from its 4-aligned start
__device__ __forceinline__ int red_tiles_of(int s0, int s1) {
  return s1 > s0 ? (s1 - (s0 & ~3) + RED_TILE - 1) / RED_TILE : 0;
}

__global__ void __launch_bounds__(1024) sq_reduce_tile_scan_kernel(const ReduceParams p) {
  __shared__ int warp_tot[32];
  cudaGridDependencySynchronize();   // programmatic serialization behind the finalize kernel (stand-alone: no-op)
  // thread t owns the `per` consecutive sequences [t*per, (t+1)*per): one block scan in total
  const int per = (p.B + 1023) / 1024;
  const int b_lo = threadIdx.x * per, b_hi = min(p.B, b_lo + per);
  int mine = 0;
#pragma unroll 4
  for (int b = b_lo; b < b_hi; ++b) mine += red_tiles_of(p.cu[b], p.cu[b + 1]);
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
    const int n = red_tiles_of(p.cu[b], p.cu[b + 1]);
    for (int i = 0; i < n; ++i) p.tile_seq[base + i] = b;   // a handful per sequence
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

__device__ __forceinline__ int red_pad(int u) { return u + ((u >> 5) << 2); }   // float index of difference u

// c[e0+w .. e0+w+3] from the two aligned vectors that hold it (e0 % 4 == 0): q0 starts at e0 + (w & ~3).
__device__ __forceinline__ float4 red_funnel(const float4& q0, const float4& q1, int s) {
  switch (s) {
    case 0: return q0;
    case 1: return make_float4(q0.y, q0.z, q0.w, q1.x);
    case 2: return make_float4(q0.z, q0.w, q1.x, q1.y);
    default: return make_float4(q0.w, q1.x, q1.y, q1.z);
  }
}

// One tile: partial sums and the minimum window sum among the windows that start in it (see the header comment).
// `tile_in_seq` = index of the tile inside sequence b, `tile` = its slot in part_sum / part_min.  Ends with thread 0
// writing the two partials; callers synchronise before reusing s_d / sh.
template <bool HAS_TG>
__device__ __forceinline__ void red_tile_body(const ReduceParams& p, float* s_d, float (*sh)[8], int b, int tile_in_seq, int tile) {
  const int s0 = p.cu[b], s1 = p.cu[b + 1];
  const int L = s1 - s0;
  const int blk0 = (s0 & ~3) + tile_in_seq * RED_TILE;                     // first token of this tile's block, 4-aligned
  const int g0 = max(s0, blk0), g1 = min(s1, blk0 + RED_TILE);             // the tile's tokens, absolute
  const int w = min(p.window, L);
  const int n_win = L - w + 1;
  const int ta = g0 - s0;                         // first window start owned by the tile (in-sequence index)
  const int jend = min(g1 - s0, n_win);           // owned starts: [ta, jend)
  const bool has_start = ta < jend;
  const int d1 = has_start ? s0 + jend - 1 : g0;  // differences c[e+w] - c[e] are formed for e in [g0, d1)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int sh4 = w & ~3, sft = w & 3;

  float a_lp = 0.f, a_n = 0.f, a_en = 0.f, a_cf = 0.f;
  // the same for a chunk on the ragged edge of the tile, of the difference range or of the arrays: scalar loads
  auto edge_chunk = [&](int e0) -> float4 {
    float d[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int e = e0 + k;
      const bool in = e >= g0 && e < g1;
      const float cfk = in ? __ldg(p.conf + e) : 0.f;
      const float vl = in ? __ldg(p.lp + e) : 0.f;
      a_en += in ? __ldg(p.ent + e) : 0.f;
      a_cf += cfk;
      const bool valid = in && (!HAS_TG || (unsigned)__ldg(p.targets + e) < (unsigned)p.V);
      a_lp += valid ? vl : 0.f;
      a_n += valid ? 1.f : 0.f;
      d[k] = (in && e < d1) ? __ldg(p.conf + e + w) - cfk : 0.f;
    }
    return make_float4(d[0], d[1], d[2], d[3]);
  };
  constexpr int ROW = 4 * RED_THREADS;            // tokens one pass of the CTA covers
  constexpr int NB = SQ_RED_NB;                           // rows per batch: up to 5 * NB 16-byte loads in flight per thread
  // CTA-uniform row classes: 2 = inside the tile and inside the difference range (look-ahead inside the arrays),
  // 1 = inside the tile, past the difference range (the last w'-1 tokens of a sequence), 0 = ragged or empty
  auto row_class = [&](int r0) -> int {
    if (!p.vec || r0 < g0 || r0 + ROW > g1) return 0;
    if (r0 >= d1) return 1;
    return (r0 + ROW <= d1 && (long long)r0 + ROW + sh4 + 4 <= p.T) ? 2 : 0;
  };
#pragma unroll 1
  for (int rb = 0; rb < RED_CHUNKS; rb += NB) {
    int cls[NB];
    float4 vl[NB], ve[NB], vc[NB], q0[NB], q1[NB];
    int4 vt[NB];
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < NB; ++i) {                // every load of the batch first
      const int e0 = blk0 + (rb + i) * ROW + 4 * threadIdx.x;
      cls[i] = row_class(blk0 + (rb + i) * ROW);
      vl[i] = cls[i] ? __ldg(reinterpret_cast<const float4*>(p.lp + e0)) : z4;
      ve[i] = cls[i] ? __ldg(reinterpret_cast<const float4*>(p.ent + e0)) : z4;
      vc[i] = cls[i] ? __ldg(reinterpret_cast<const float4*>(p.conf + e0)) : z4;
      if (HAS_TG) vt[i] = cls[i] ? __ldg(reinterpret_cast<const int4*>(p.targets + e0)) : make_int4(-1, -1, -1, -1);
      q0[i] = (cls[i] == 2) ? __ldg(reinterpret_cast<const float4*>(p.conf + e0 + sh4)) : z4;
      // the vector after q0 is the next lane's q0: only lane 31 has to load it
      q1[i] = (cls[i] == 2 && sft && lane == 31) ? __ldg(reinterpret_cast<const float4*>(p.conf + e0 + sh4 + 4)) : z4;
    }
#pragma unroll
    for (int i = 0; i < NB; ++i) {
      const int c = (rb + i) * RED_THREADS + threadIdx.x;
      float4 dv = z4;
      if (cls[i]) {
        a_en += (ve[i].x + ve[i].y) + (ve[i].z + ve[i].w);
        a_cf += (vc[i].x + vc[i].y) + (vc[i].z + vc[i].w);
        if (HAS_TG) {
          const bool k0 = (unsigned)vt[i].x < (unsigned)p.V, k1 = (unsigned)vt[i].y < (unsigned)p.V;
          const bool k2 = (unsigned)vt[i].z < (unsigned)p.V, k3 = (unsigned)vt[i].w < (unsigned)p.V;
          a_lp += ((k0 ? vl[i].x : 0.f) + (k1 ? vl[i].y : 0.f)) + ((k2 ? vl[i].z : 0.f) + (k3 ? vl[i].w : 0.f));
          a_n += (float)((int)k0 + (int)k1 + (int)k2 + (int)k3);
        } else {
          a_lp += (vl[i].x + vl[i].y) + (vl[i].z + vl[i].w);
          a_n += 4.f;
        }
        if (cls[i] == 2) {
          if (sft) {                              // CTA-uniform
            const float nx = __shfl_down_sync(0xffffffffu, q0[i].x, 1);
            const float ny = __shfl_down_sync(0xffffffffu, q0[i].y, 1);
            const float nz = __shfl_down_sync(0xffffffffu, q0[i].z, 1);
            if (lane != 31) q1[i] = make_float4(nx, ny, nz, 0.f);
          }
          const float4 ah = red_funnel(q0[i], q1[i], sft);
          dv = make_float4(ah.x - vc[i].x, ah.y - vc[i].y, ah.z - vc[i].z, ah.w - vc[i].w);
        }
      } else {
        const int row0 = blk0 + (rb + i) * ROW;
        if (row0 + ROW > g0 && row0 < g1) dv = edge_chunk(blk0 + 4 * c);
      }
      *reinterpret_cast<float4*>(s_d + red_pad(4 * c)) = dv;
    }
  }
  float a_s0 = 0.f;                               // S(ta), summed directly
  if (has_start)
    for (int i = threadIdx.x; i < w; i += RED_THREADS) a_s0 += __ldg(p.conf + g0 + i);
  a_lp = warp_sum(a_lp); a_n = warp_sum(a_n); a_en = warp_sum(a_en); a_cf = warp_sum(a_cf); a_s0 = warp_sum(a_s0);
  __syncthreads();

  // each thread scans its 32 consecutive differences, then one block scan of the 256 totals
  const int uv0 = g0 - blk0, uv1 = d1 - blk0;     // differences that stand for a window start: u in [uv0, uv1)
  const int ub = threadIdx.x * RED_PER_THREAD;
  float run = 0.f, tmin = CUDART_INF_F;
  if (ub < uv1 && ub + RED_PER_THREAD > uv0) {
    const float4* q = reinterpret_cast<const float4*>(s_d + red_pad(ub));
    const bool full = ub >= uv0 && ub + RED_PER_THREAD <= uv1;
#pragma unroll
    for (int i = 0; i < RED_PER_THREAD / 4; ++i) {
      const float4 v = q[i];
      const float x[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        run += x[k];
        const int u = ub + 4 * i + k;
        if (full || (u >= uv0 && u < uv1)) tmin = fminf(tmin, run);
      }
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
  for (int qq = 0; qq < warp; ++qq) woff += sh[qq][5];
  float wmin = tmin + (woff + incl - run);        // +inf stays +inf for threads without a window
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) wmin = fminf(wmin, __shfl_xor_sync(0xffffffffu, wmin, off));
  if (lane == 0) sh[warp][4] = wmin;
  __syncthreads();
  if (threadIdx.x == 0) {
    float s_lp = 0.f, s_n = 0.f, s_en = 0.f, s_cf = 0.f, sa = 0.f, best = 0.f;   // 0: the start ta itself
    for (int qq = 0; qq < RED_WARPS; ++qq) {      // fixed order: deterministic
      s_lp += sh[qq][0]; s_n += sh[qq][1]; s_en += sh[qq][2]; s_cf += sh[qq][3]; sa += sh[qq][6];
      best = fminf(best, sh[qq][4]);
    }
    p.part_sum[tile] = make_float4(s_lp, s_n, s_en, s_cf);
    p.part_min[tile] = has_start ? sa + best : CUDART_INF_F;
  }
}

template <bool HAS_TG>
__global__ void __launch_bounds__(RED_THREADS) sq_reduce_tile_part_kernel(const ReduceParams p) {
  extern __shared__ __align__(16) float s_d[];   // window-sum differences of the block, padded
  __shared__ float sh[RED_WARPS][8];
  cudaGridDependencySynchronize();               // launched with programmatic serialization behind tile_scan
  const int tile = blockIdx.x;
  if (tile >= p.tile_base[p.B]) return;
  const int b = p.tile_seq[tile];
  red_tile_body<HAS_TG>(p, s_d, sh, b, tile - p.tile_base[b], tile);
}

// Fold of one sequence's tile partials [t0, t1) by one warp, fixed order, fp64 accumulators.
__device__ __forceinline__ void red_fold_sequence(const ReduceParams& p, int b, int L, int t0, int t1, int lane) {
  double s_lp = 0.0, s_n = 0.0, s_en = 0.0, s_cf = 0.0;
  float best = CUDART_INF_F;
  for (int t = t0 + lane; t < t1; t += 32) {
    const float4 v = __ldcg(p.part_sum + t);
    s_lp += v.x; s_n += v.y; s_en += v.z; s_cf += v.w;
    best = fminf(best, __ldcg(p.part_min + t));
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

__global__ void __launch_bounds__(128) sq_reduce_seq_final_kernel(const ReduceParams p) {
  cudaGridDependencySynchronize();               // launched with programmatic serialization behind tile_part
  const int b = blockIdx.x * 4 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (b >= p.B) return;
  const int L = p.cu[b + 1] - p.cu[b];
  if (L <= 0) return;                            // tile_scan already wrote the NaNs
  red_fold_sequence(p, b, L, p.tile_base[b], p.tile_base[b + 1], lane);
}

// Single-launch form (B <= RED_FUSED_MAX_SEQS): every CTA rebuilds the tile table in shared memory (a block scan over
// the B sequence lengths: 16 KB of L2-resident cu_seqlens at B = 4096, ~2 us, instead of a one-CTA launch), takes
// tiles round-robin, and the CTA that finishes a sequence's LAST tile folds that sequence's partials in fixed order
// (fence + atomic counter, reset by the folder, so the counters are all zero again when the kernel ends).  Used when
// the whole problem is one wave of CTAs (the scoring pipeline: a few dozen tiles), where it replaces three
// latency-bound launches by one; on large inputs the three-launch form is 2x faster (a persistent CTA pays fence +
// atomic + barriers per tile in series) and is kept.  Results are bit-identical to the three-launch form.
constexpr int RED_FUSED_MAX_SEQS = 12287;   // (B + 1) ints of shared memory next to the difference array

template <bool HAS_TG>
__global__ void __launch_bounds__(RED_THREADS) sq_reduce_fused_kernel(const ReduceParams p) {
  extern __shared__ __align__(16) float s_d[];
  __shared__ float sh[RED_WARPS][8];
  __shared__ int s_warp[RED_WARPS];
  __shared__ int s_carry, s_last;
  int* tb = reinterpret_cast<int*>(s_d + RED_SMEM_BYTES / 4);   // [B+1] exclusive scan of the tiles per sequence
  cudaGridDependencySynchronize();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int base = 0; base < p.B; base += RED_THREADS) {
    const int b = base + threadIdx.x;
    const int n = b < p.B ? red_tiles_of(__ldg(p.cu + b), __ldg(p.cu + b + 1)) : 0;
    int x = n;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, x, off);
      if (lane >= off) x += y;
    }
    if (lane == 31) s_warp[warp] = x;
    __syncthreads();
    int woff = s_carry;
    for (int q = 0; q < warp; ++q) woff += s_warp[q];
    if (b < p.B) {
      tb[b] = woff + x - n;
      if (n == 0 && (b % gridDim.x) == blockIdx.x) {   // empty sequence: exactly one CTA writes its NaNs
        const float nan = CUDART_NAN_F;
        p.out_lp[b] = nan; p.out_ent[b] = nan; p.out_conf[b] = nan; p.out_min[b] = nan;
      }
    }
    __syncthreads();
    if (threadIdx.x == RED_THREADS - 1) s_carry = woff + x;
    __syncthreads();
  }
  const int total = s_carry;
  if (threadIdx.x == 0) tb[p.B] = total;
  __syncthreads();
  for (int tile = blockIdx.x; tile < total; tile += gridDim.x) {
    int lo = 0, hi = p.B - 1;                     // the sequence b with tb[b] <= tile < tb[b+1]
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (tb[mid] <= tile) lo = mid; else hi = mid - 1;
    }
    const int b = lo;
    red_tile_body<HAS_TG>(p, s_d, sh, b, tile - tb[b], tile);
    if (threadIdx.x == 0) {
      __threadfence();                            // the partials above are visible before the count
      const int done = atomicAdd(p.seq_done + b, 1) + 1;
      s_last = (done == tb[b + 1] - tb[b]) ? 1 : 0;
    }
    __syncthreads();
    if (s_last && warp == 0) {
      __threadfence();
      red_fold_sequence(p, b, __ldg(p.cu + b + 1) - __ldg(p.cu + b), tb[b], tb[b + 1], lane);
      if (lane == 0) p.seq_done[b] = 0;
    }
    __syncthreads();                              // s_d / sh / s_last are reused by the next tile
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Streaming form (large inputs; RS_WMIN <= window <= RS_WMAX; 16-byte aligned arrays): two launches.
//
// The tile forms above cut tiles at sequence starts, so a CTA must know its sequence before it can load anything
// (table lookup or search -> loads -> arithmetic, every step a dependent round trip through a saturated memory system),
// and a CTA's lifetime is mostly latency.  Here the streaming kernel does not look at cu_seqlens at all:
//   stream : CTA x owns the FIXED block [x * TB, (x+1) * TB) of the packed arrays (TB = 4096 or 6144), warp q its range of R = TB / 16 tokens.
//            1. every thread issues all its 16-byte loads at once (lp, ent, conf, targets of its 8 tokens + one vector
//               of the look-ahead range [block end, block end + w)): one round trip;
//            2. exclusive prefix sums P of conf over block + look-ahead: in registers (per vector, per warp by
//               shuffles), one barrier for the 32 warp totals, then P goes to shared memory;
//            3. window sums S(j) = P[j + w] - P[j] straight from shared memory; the prefix restarts in every block, so
//               fp32 error does not grow with the sequence;
//            4. one record per range, whatever sequences it touches: the four sums over its 256 tokens, the minimum of
//               S(j) over its 256 window starts, and S at its first token.
//   fold   : one warp per sequence.  Ranges that lie inside the sequence contribute their records (sums; the minimum
//            where all 256 windows end inside the sequence).  What is left is at most one ragged range at each end of
//            the sequence and of its window starts: those tokens are read again (<= 512 per array and sequence, from
//            L2), and the window sums of a ragged range are rebuilt from the range's recorded first sum by a scan of
//            the differences c[m + w] - c[m].  fp64 accumulators, fixed order: deterministic.  Empty sequences get
//            NaNs; a sequence shorter than the window has one window, itself: min = mean conf.
// The prefix runs across sequence boundaries inside a block, so a non-finite conf value spoils the window sums of its
// whole 4096-token block (the tile forms confine it to its sequence); c(i) of Eq. 3 is always finite.
constexpr int RS_THREADS = 512;
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_WMAX = 2048;       // widest window: the look-ahead is one 16-byte vector per thread
constexpr int RS_WMIN = 128;        // narrowest: S(j) = P[j+w] - P[j] with P up to ~6144 x mean(conf) in fp32; the rounding of P
                                    // (~1e-7 relative to P, i.e. ~5e-6 of a 128-element sum) would reach 1e-3 of a 1-element one

__device__ __forceinline__ float4 rs_load4(const float* a, int e, int T) {   // elements at or past T read as 0
  if (e + 4 <= T) return __ldg(reinterpret_cast<const float4*>(a + e));
  float4 v;
  v.x = e < T ? __ldg(a + e) : 0.f;         v.y = e + 1 < T ? __ldg(a + e + 1) : 0.f;
  v.z = e + 2 < T ? __ldg(a + e + 2) : 0.f; v.w = e + 3 < T ? __ldg(a + e + 3) : 0.f;
  return v;
}
__device__ __forceinline__ int4 rs_load4i(const int32_t* a, int e, int T) {  // ... as -1
  if (e + 4 <= T) return __ldg(reinterpret_cast<const int4*>(a + e));
  int4 v;
  v.x = e < T ? __ldg(a + e) : -1;         v.y = e + 1 < T ? __ldg(a + e + 1) : -1;
  v.z = e + 2 < T ? __ldg(a + e + 2) : -1; v.w = e + 3 < T ? __ldg(a + e + 3) : -1;
  return v;
}
// inclusive scan over the lanes of a warp
__device__ __forceinline__ float rs_warp_incl(float x, int lane) {
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const float y = __shfl_up_sync(0xffffffffu, x, off);
    if (lane >= off) x += y;
  }
  return x;
}
// minimum over the warp in one instruction (sm_100a: redux.sync on f32; the inputs are finite or +inf)
__device__ __forceinline__ float rs_warp_min(float v) {
  float r;
  asm volatile("redux.sync.min.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
  return r;
}
// Sums of four values over the warp in 6 shuffles instead of 20: lanes trade halves of the value set while they fold
// (xor 16: keep two of four, xor 8: keep one of two, then three plain steps).  Returns the total of a in lanes 0..7,
// of b in lanes 8..15, of c in lanes 16..23, of d in lanes 24..31.
__device__ __forceinline__ float rs_warp_sum4(float a, float b, float c, float d, int lane) {
  const bool hi = lane & 16;
  const float k0 = hi ? c : a, k1 = hi ? d : b;              // kept
  const float g0 = hi ? a : c, g1 = hi ? b : d;              // given away
  const float x0 = k0 + __shfl_xor_sync(0xffffffffu, g0, 16);
  const float x1 = k1 + __shfl_xor_sync(0xffffffffu, g1, 16);
  const bool h8 = lane & 8;
  float y = (h8 ? x1 : x0) + __shfl_xor_sync(0xffffffffu, h8 ? x0 : x1, 8);
  y += __shfl_xor_sync(0xffffffffu, y, 4);
  y += __shfl_xor_sync(0xffffffffu, y, 2);
  y += __shfl_xor_sync(0xffffffffu, y, 1);
  return y;
}

// NV = 16-byte vectors per lane and array: a warp's range is R = 128 NV tokens, a CTA's block 16 R.  More bytes per thread
// in flight beat more threads: with targets (four arrays) NV = 2 at two CTAs per SM streams at 0.96 of the copy peak, without
// them NV = 3 at two CTAs (NV = 2 at three CTAs: 0.91).
template <int NV> struct RsCfg {
  static constexpr int R = 128 * NV;           // tokens per warp = per record
  static constexpr int TB = RS_WARPS * R;      // tokens per CTA
};

template <bool HAS_TG, int NV>
__global__ void __launch_bounds__(RS_THREADS, 2) sq_reduce_stream_kernel(const ReduceParams p) {
  constexpr int R = RsCfg<NV>::R, TB = RsCfg<NV>::TB;
  __shared__ __align__(16) float s_P[TB + RS_WMAX + 4];      // exclusive prefix of conf over block + look-ahead
  __shared__ float s_tot[32];                                // totals: 16 warp ranges, then 16 look-ahead runs of 128
  cudaGridDependencySynchronize();
  cudaTriggerProgrammaticLaunchCompletion();                 // the fold kernel may start its record-independent part
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int T = (int)p.T;                                    // the host takes this form only when T + TB + RS_WMAX fits an int
  const int blk0 = blockIdx.x * TB;
  const int e0 = blk0 + warp * R + 4 * lane;                 // lane l owns tokens e0 + 128 k .. + 3, k < NV, of the warp's range
  const int ela = blk0 + TB + 4 * threadIdx.x;
  const int w = p.window;
  const bool has_la = 4 * (int)threadIdx.x < w;

  // 1. every load first
  float4 vl[NV], ve[NV], vc[NV];
  int4 vt[NV];
  float4 la = make_float4(0.f, 0.f, 0.f, 0.f);
  if (blk0 + TB + RS_WMAX <= T) {                            // CTA-uniform: no vector crosses the end of the arrays
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      vl[k] = __ldg(reinterpret_cast<const float4*>(p.lp + e0 + 128 * k));
      ve[k] = __ldg(reinterpret_cast<const float4*>(p.ent + e0 + 128 * k));
      vc[k] = __ldg(reinterpret_cast<const float4*>(p.conf + e0 + 128 * k));
      if (HAS_TG) vt[k] = __ldg(reinterpret_cast<const int4*>(p.targets + e0 + 128 * k));
    }
    if (has_la) la = __ldg(reinterpret_cast<const float4*>(p.conf + ela));
  } else {
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      vl[k] = rs_load4(p.lp, e0 + 128 * k, T);
      ve[k] = rs_load4(p.ent, e0 + 128 * k, T);
      vc[k] = rs_load4(p.conf, e0 + 128 * k, T);
      if (HAS_TG) vt[k] = rs_load4i(p.targets, e0 + 128 * k, T);
    }
    if (has_la) la = rs_load4(p.conf, ela, T);
  }

  // 2. prefix sums of conf: per vector, per warp, per block
  float own_excl[NV], t_cf = 0.f;
  {
    float before = 0.f;                                      // sum of the vectors k' < k of this warp's range
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      const float t = (vc[k].x + vc[k].y) + (vc[k].z + vc[k].w);
      const float inc = rs_warp_incl(t, lane);
      own_excl[k] = before + (inc - t);
      before += __shfl_sync(0xffffffffu, inc, 31);
      t_cf += t;
    }
    const float la_t = (la.x + la.y) + (la.z + la.w);
    const float la_incl = rs_warp_incl(la_t, lane);
    if (lane == 31) { s_tot[warp] = before; s_tot[RS_WARPS + warp] = la_incl; }
    la.w = la_incl - la_t;                                   // la.w is not needed below: the slot carries the exclusive prefix
  }
  __syncthreads();
  {
    const float t = s_tot[lane];
    const float ex = rs_warp_incl(t, lane) - t;
    const float off_own = __shfl_sync(0xffffffffu, ex, warp);
    const float off_la = __shfl_sync(0xffffffffu, ex, RS_WARPS + warp);
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      const float b0 = off_own + own_excl[k];
      float4 o;
      o.x = b0; o.y = b0 + vc[k].x; o.z = o.y + vc[k].y; o.w = o.z + vc[k].z;
      *reinterpret_cast<float4*>(s_P + warp * R + k * 128 + 4 * lane) = o;
    }
    const float b0 = off_la + la.w;
    float4 o;
    o.x = b0; o.y = b0 + la.x; o.z = o.y + la.y; o.w = o.z + la.z;
    *reinterpret_cast<float4*>(s_P + TB + 4 * threadIdx.x) = o;
  }
  // the lane's sums, while the barrier fills
  float a_en = 0.f, a_lp = 0.f, a_n = 0.f;
#pragma unroll
  for (int k = 0; k < NV; ++k) {
    a_en += (ve[k].x + ve[k].y) + (ve[k].z + ve[k].w);
    if (HAS_TG) {
      const bool k0 = (unsigned)vt[k].x < (unsigned)p.V, k1 = (unsigned)vt[k].y < (unsigned)p.V;
      const bool k2 = (unsigned)vt[k].z < (unsigned)p.V, k3 = (unsigned)vt[k].w < (unsigned)p.V;
      a_lp += ((k0 ? vl[k].x : 0.f) + (k1 ? vl[k].y : 0.f)) + ((k2 ? vl[k].z : 0.f) + (k3 ? vl[k].w : 0.f));
      a_n += (float)((int)k0 + (int)k1 + (int)k2 + (int)k3);
    } else {
      a_lp += (vl[k].x + vl[k].y) + (vl[k].z + vl[k].w);
      a_n += 4.f;
    }
  }
  const float tot = rs_warp_sum4(a_lp, a_n, a_en, t_cf, lane);
  __syncthreads();

  // 3. the R window sums that start in this range
  const float* Pl = s_P + warp * R + 4 * lane;
  float mn = CUDART_INF_F, s_first = 0.f;
  if ((w & 3) == 0) {                                        // 16-byte shared loads line up
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      const float4 lo = *reinterpret_cast<const float4*>(Pl + 128 * k);
      const float4 hi = *reinterpret_cast<const float4*>(Pl + 128 * k + w);
      if (k == 0) s_first = hi.x - lo.x;
      mn = fminf(mn, fminf(fminf(hi.x - lo.x, hi.y - lo.y), fminf(hi.z - lo.z, hi.w - lo.w)));
    }
  } else {
#pragma unroll
    for (int k = 0; k < NV; ++k)
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float sj = Pl[128 * k + i + w] - Pl[128 * k + i];
        if (k == 0 && i == 0) s_first = sj;
        mn = fminf(mn, sj);
      }
  }
  mn = rs_warp_min(mn);
  // 4. the record of this range
  const int range = blockIdx.x * RS_WARPS + warp;
  if ((lane & 7) == 0) reinterpret_cast<float*>(p.part_sum + range)[lane >> 3] = tot;
  if (lane == 0) reinterpret_cast<float2*>(p.part_min)[range] = make_float2(mn, s_first);
}

// Window sums of a ragged range r (tokens [R r, R r + R)) are rebuilt from its recorded first sum S(R r):
// S(j + 1) = S(j) + c[j + w] - c[j].  Lane l rebuilds the starts R r + PL l .. + PL - 1 (PL = R / 32); only starts in [lo, hi) count.
template <int PL> struct RsRagged {
  float d[PL];    // d[i] = S(m0 + i + 1) - S(m0 + i)
  float excl;     // S(m0) - S(R r)
  int m0, lo, hi; // lo >= hi: nothing to do
};
template <int PL>
__device__ __forceinline__ void rs_ragged_load(RsRagged<PL>& g, const ReduceParams& p, int r, int lo, int hi, int w, int lane) {
  g.m0 = r * (32 * PL) + PL * lane; g.lo = lo; g.hi = hi;
  float run = 0.f;
#pragma unroll
  for (int i = 0; i < PL; ++i) {                             // only differences below the last start matter
    const int m = g.m0 + i;
    g.d[i] = (m + 1 < hi) ? __ldg(p.conf + m + w) - __ldg(p.conf + m) : 0.f;   // m + w < hi + w - 1 <= s1 - 1: inside the arrays
    run += g.d[i];
  }
  g.excl = rs_warp_incl(run, lane) - run;
}
template <int PL>
__device__ __forceinline__ float rs_ragged_min(const RsRagged<PL>& g, float s_range_first) {
  float s = s_range_first + g.excl, best = CUDART_INF_F;
#pragma unroll
  for (int i = 0; i < PL; ++i) {
    if (g.m0 + i >= g.lo && g.m0 + i < g.hi) best = fminf(best, s);
    s += g.d[i];
  }
  return best;
}

// One warp per sequence.  Everything that does not depend on the stream kernel's records -- cu_seqlens, the ragged
// ends of the sequence, the differences of the ragged window ranges -- is read BEFORE the grid dependency wait, i.e.
// underneath the stream kernel's last wave (the stream kernel triggers this launch early; it does so after its own
// dependency wait, so whatever produced lp / ent / conf has completed by the time this kernel can start).
template <int NV>
__global__ void __launch_bounds__(128) sq_reduce_stream_fold_kernel(const ReduceParams p) {
  constexpr int R = RsCfg<NV>::R, PL = R / 32;
  const int b = blockIdx.x * 4 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  // Every warp waits for the stream kernel before it leaves, also those with nothing to fold: a fold grid that finished
  // without waiting (every sequence empty) would leave "this kernel is complete => the stream kernel is complete" to
  // unspecified behaviour of programmatic launches, and the stream kernel still writes the ctx's records.
  if (b >= p.B) { cudaGridDependencySynchronize(); return; }
  const int s0 = __ldg(p.cu + b), s1 = __ldg(p.cu + b + 1);
  const int L = s1 - s0, w = p.window;
  if (L <= 0) {
    if (lane == 0) { const float nan = CUDART_NAN_F; p.out_lp[b] = nan; p.out_ent[b] = nan; p.out_conf[b] = nan; p.out_min[b] = nan; }
    cudaGridDependencySynchronize();
    return;
  }
  // sums: the ranges [r_a, r_b) lie inside the sequence; what is left of it are the tokens [s0, h1) and [t0, s1)
  const int r_a = (s0 + R - 1) / R, r_b = s1 / R;
  const int h1 = r_a < r_b ? r_a * R : s1, t0 = r_a < r_b ? r_b * R : s1;
  double s_lp = 0.0, s_n = 0.0, s_en = 0.0, s_cf = 0.0;
  // the ragged ends, fewer than R tokens each (2 R when no range lies inside the sequence): every load of a pass at once
  auto raw = [&](int e_lo, int e_hi) {
    for (int base = e_lo; base < e_hi; base += 256) {
      float xl[8], xe[8], xc[8];
      int xt[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int e = base + lane + 32 * i;
        const bool in = e < e_hi;
        xl[i] = in ? __ldg(p.lp + e) : 0.f;
        xe[i] = in ? __ldg(p.ent + e) : 0.f;
        xc[i] = in ? __ldg(p.conf + e) : 0.f;
        xt[i] = in ? (p.targets ? __ldg(p.targets + e) : 0) : -1;
      }
      float f_lp = 0.f, f_n = 0.f, f_en = 0.f, f_cf = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const bool valid = (unsigned)xt[i] < (unsigned)p.V;
        f_lp += valid ? xl[i] : 0.f;
        f_n += valid ? 1.f : 0.f;
        f_en += xe[i];
        f_cf += xc[i];
      }
      s_lp += f_lp; s_n += f_n; s_en += f_en; s_cf += f_cf;
    }
  };
  raw(s0, h1);
  raw(t0, s1);
  // window starts [s0, jl]: the ranges [r_a, r_c) hold only valid starts; a ragged range at each end
  const int jl = s1 - w;
  const int r_c = (L >= w) ? (jl + 1) / R : r_a;
  const int r_t = max(r_c, r_a);
  RsRagged<PL> gh, gt;
  gh.lo = gh.hi = gt.lo = gt.hi = 0;
  if (L >= w && (s0 % R)) rs_ragged_load(gh, p, s0 / R, s0, min(jl + 1, r_a * R), w, lane);
  if (L >= w && r_t * R <= jl) rs_ragged_load(gt, p, r_t, r_t * R, jl + 1, w, lane);

  cudaGridDependencySynchronize();                           // the records
  for (int r = r_a + lane; r < r_b; r += 32) {
    const float4 v = __ldcg(p.part_sum + r);
    s_lp += v.x; s_n += v.y; s_en += v.z; s_cf += v.w;
  }
  float best = CUDART_INF_F;
  for (int r = r_a + lane; r < r_c; r += 32) best = fminf(best, __ldcg(p.part_min + 2 * r));
  if (gh.lo < gh.hi) best = fminf(best, rs_ragged_min(gh, __ldcg(p.part_min + 2 * (s0 / R) + 1)));
  if (gt.lo < gt.hi) best = fminf(best, rs_ragged_min(gt, __ldcg(p.part_min + 2 * r_t + 1)));
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    s_lp += __shfl_xor_sync(0xffffffffu, s_lp, off);
    s_n += __shfl_xor_sync(0xffffffffu, s_n, off);
    s_en += __shfl_xor_sync(0xffffffffu, s_en, off);
    s_cf += __shfl_xor_sync(0xffffffffu, s_cf, off);
    best = fminf(best, __shfl_xor_sync(0xffffffffu, best, off));
  }
  if (lane == 0) {
    p.out_lp[b] = (s_n > 0.0) ? (float)(s_lp / s_n) : CUDART_NAN_F;
    p.out_ent[b] = (float)(s_en / (double)L);
    p.out_conf[b] = (float)(s_cf / (double)L);
    p.out_min[b] = (L >= w) ? best / (float)w : (float)(s_cf / (double)L);
  }
}

}  // namespace sq
