// sq_route_kernel.cuh -- SURVEY section 8(f)-1: from one scalar per trajectory to a routing decision,
// on the device, with no host round trip.
//
//   GC(g)   = (1/K) sum_{tau in g} C(tau)                                   Eq. 4 (right)
//   theta_q = Percentile_p({GC(g) : g in G_q \ B_lite})                     Eq. 6
//             (linear interpolation between order statistics at rank p/100 * (n-1); reading #13)
//   mu(g,q) = Model 1 if GC(g) > theta_q ("easy", strict) else Model 2      Eq. 7
//   select  : P(i) = exp(f_i / zeta) / sum_j exp(f_j / zeta) per problem
//
// One CTA per problem.  The comparison GC > theta decides an integer; it is taken in fp32 on the GC and theta this
// kernel REPORTS (_rn intrinsics: no FMA contraction, so the reported values are the compared ones), and the parity
// test judges it against the fp64 definition with a derived fp32 margin.  Codes: 0 = B_lite (caller-supplied mask),
// 1 = Model 1, 2 = Model 2, 3 = GC not finite (the group holds an empty trajectory, C(tau) = NaN: it takes no part in
// the percentile, reading #24), -1 = the problem has more groups than the sort holds (theta = NaN).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace sq {

constexpr int ROUTE_THREADS = 256;
constexpr int ROUTE_MAX_GROUPS = 1024;   // groups per problem the shared-memory sort holds

struct RouteParams {
  const float* seq_conf;          // [N] C(tau)
  const int32_t* group_members;   // [G][K] indices into seq_conf
  const int32_t* group_offsets;   // [Q+1]
  const uint8_t* lite_mask;       // [G] or null
  int K;
  float percentile;
  float* group_fitness;           // [G]
  float* theta;                   // [Q]
  int32_t* route;                 // [G]
};

__global__ void __launch_bounds__(ROUTE_THREADS) sq_route_kernel(const RouteParams p) {
  __shared__ float sv[ROUTE_MAX_GROUPS];
  __shared__ int s_n;
  __shared__ float s_theta;
  const int q = blockIdx.x;
  const int g0 = p.group_offsets[q], g1 = p.group_offsets[q + 1];
  const int ng = g1 - g0;
  if (ng > ROUTE_MAX_GROUPS) {   // the host-side bound was wrong: flag the problem instead of routing on a partial sort
    for (int i = threadIdx.x; i < ng; i += ROUTE_THREADS) p.route[g0 + i] = -1;
    if (threadIdx.x == 0) p.theta[q] = CUDART_NAN_F;
    return;
  }
  if (threadIdx.x == 0) s_n = 0;
  __syncthreads();
  int live = 0;
  for (int i = threadIdx.x; i < ROUTE_MAX_GROUPS; i += ROUTE_THREADS) {
    float key = CUDART_INF_F;
    if (i < ng) {
      const int g = g0 + i;
      float acc = 0.f;
      for (int j = 0; j < p.K; ++j) acc = __fadd_rn(acc, p.seq_conf[p.group_members[(size_t)g * p.K + j]]);
      const float gc = __fdiv_rn(acc, (float)p.K);
      p.group_fitness[g] = gc;
      const bool lite = p.lite_mask && p.lite_mask[g];
      if (!lite && isfinite(gc)) { key = gc; ++live; }   // a NaN would break the sort's order
    }
    sv[i] = key;
  }
  atomicAdd(&s_n, live);
  __syncthreads();
  // bitonic sort, ascending; lite groups and padding are +inf and end up behind the n live values
  for (int k = 2; k <= ROUTE_MAX_GROUPS; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < ROUTE_MAX_GROUPS; i += ROUTE_THREADS) {
        const int ixj = i ^ j;
        if (ixj > i) {
          const float a = sv[i], b = sv[ixj];
          const bool up = (i & k) == 0;
          if ((a > b) == up) { sv[i] = b; sv[ixj] = a; }
        }
      }
      __syncthreads();
    }
  }
  if (threadIdx.x == 0) {
    const int n = s_n;
    float th = CUDART_NAN_F;
    if (n > 0) {
      const float pos = __fmul_rn(__fdiv_rn(p.percentile, 100.f), (float)(n - 1));
      const int lo = (int)floorf(pos);
      const int hi = min(lo + 1, n - 1);
      const float frac = __fsub_rn(pos, (float)lo);
      th = __fadd_rn(sv[lo], __fmul_rn(frac, __fsub_rn(sv[hi], sv[lo])));
    }
    s_theta = th;
    p.theta[q] = th;
  }
  __syncthreads();
  const float th = s_theta;
  for (int i = threadIdx.x; i < ng; i += ROUTE_THREADS) {
    const int g = g0 + i;
    const bool lite = p.lite_mask && p.lite_mask[g];
    const float gc = p.group_fitness[g];
    p.route[g] = lite ? 0 : (!isfinite(gc) ? 3 : (gc > th ? 1 : 2));
  }
}

struct SelectParams {
  const float* fitness;        // [N]
  const int32_t* pop_offsets;  // [Q+1]
  float inv_zeta;
  float* prob;                 // [N]
};

__global__ void __launch_bounds__(ROUTE_THREADS) sq_select_prob_kernel(const SelectParams p) {
  __shared__ float red[ROUTE_THREADS / 32];
  __shared__ float s_bcast;
  const int q = blockIdx.x;
  const int i0 = p.pop_offsets[q], i1 = p.pop_offsets[q + 1];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float m = -CUDART_INF_F;
  for (int i = i0 + threadIdx.x; i < i1; i += ROUTE_THREADS) m = fmaxf(m, p.fitness[i]);
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, off));
  if (lane == 0) red[warp] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    float v = red[0];
    for (int w = 1; w < ROUTE_THREADS / 32; ++w) v = fmaxf(v, red[w]);
    s_bcast = v;
  }
  __syncthreads();
  m = s_bcast;
  float s = 0.f;
  for (int i = i0 + threadIdx.x; i < i1; i += ROUTE_THREADS) s += expf((p.fitness[i] - m) * p.inv_zeta);
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  __syncthreads();
  if (lane == 0) red[warp] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    float v = 0.f;
    for (int w = 0; w < ROUTE_THREADS / 32; ++w) v += red[w];   // fixed order
    s_bcast = v;
  }
  __syncthreads();
  const float inv = 1.f / s_bcast;
  for (int i = i0 + threadIdx.x; i < i1; i += ROUTE_THREADS) p.prob[i] = expf((p.fitness[i] - m) * p.inv_zeta) * inv;
}

}  // namespace sq
