// sq_finalize_kernel.cuh -- step a6: merge the vocab-chunk partial states of every row and finalise.
//
//   lse = M + ln S,  M = max_c m_c,  S = sum_c s_c e^{m_c - M}      (merged in fp64)
//   entropy = ln S - U / S,  U = sum_c e^{m_c - M} (u_c + (m_c - M) s_c)
//   target_logprob = z_target - lse
//   topk_logprob_j = z_(j) - lse,  conf = c(i) = -(1/k) sum_j topk_logprob_j    (Eq. 3)
//
// One warp per token row; lane c holds chunk c's state (num_chunks <= 32).  The running max / sum /
// entropy merge is a warp-shuffle reduction; the top-k merge is k rounds of a warp arg-max over the
// heads of the per-chunk sorted lists (ties: larger value first, then smaller vocabulary id).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sq {

struct FinalizeParams {
  int T, V, k, cap, num_chunks;
  const int32_t* targets;
  const float* part_m;
  const float* part_s;
  const float* part_u;
  const float* part_cs;     // Kahan residues of s and u
  const float* part_cu;
  const float* part_topv;   // [C][cap][T]
  const int32_t* part_topi;
  const float* zt;
  float* lse;
  float* target_logprob;
  float* entropy;
  float* conf;
  float* topk_logprob;      // [T][k] or null
  int32_t* topk_index;      // [T][k] or null
};

constexpr int FIN_WARPS = 8;

__global__ void __launch_bounds__(FIN_WARPS * 32)
sq_finalize_kernel(const FinalizeParams p) {
  const int lane = threadIdx.x & 31;
  const int row = blockIdx.x * FIN_WARPS + (threadIdx.x >> 5);
  if (row >= p.T) return;
  const unsigned FULL = 0xffffffffu;
  const float NEG = -1.0e30f;
  const bool has = lane < p.num_chunks;
  const size_t o = (size_t)lane * p.T + row;
  const float m_c = has ? p.part_m[o] : NEG;
  // the merge runs in fp64: S - 1 of a peaked row is ~1e-4 and carries the whole entropy
  const double s_c = has ? ((double)p.part_s[o] - (double)p.part_cs[o]) : 0.0;
  const double u_c = has ? ((double)p.part_u[o] - (double)p.part_cu[o]) : 0.0;

  float M = m_c;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) M = fmaxf(M, __shfl_xor_sync(FULL, M, off));
  const double dm = (double)m_c - (double)M;
  const double w = has ? exp(dm) : 0.0;
  double S = w * s_c;
  double U = w * (u_c + dm * s_c);
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    S += __shfl_xor_sync(FULL, S, off);
    U += __shfl_xor_sync(FULL, U, off);
  }
  const double lnS = log(S);
  const float lse = (float)((double)M + lnS);

  // ---- top-k merge: lane c walks chunk c's descending list
  int pos = 0;
  float hv = NEG; int hi = 0x7fffffff;
  auto load_head = [&]() {
    if (has && pos < p.cap) {
      const size_t oj = ((size_t)lane * p.cap + pos) * p.T + row;
      hv = p.part_topv[oj];
      hi = p.part_topi[oj];
      if (hi < 0) { hv = NEG; hi = 0x7fffffff; }   // unfilled slot
    } else {
      hv = NEG; hi = 0x7fffffff;
    }
  };
  load_head();
  float acc = 0.f;       // sum of the k best logits
  float my_v = 0.f; int my_i = 0;   // lane j keeps the j-th winner for a coalesced store
  for (int j = 0; j < p.k; ++j) {
    float bv = hv; int bi = hi;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const float ov = __shfl_xor_sync(FULL, bv, off);
      const int oi = __shfl_xor_sync(FULL, bi, off);
      if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    acc += bv;
    if (lane == j) { my_v = bv; my_i = bi; }
    if (hi == bi && hv == bv) { ++pos; load_head(); }   // vocabulary ids are unique: exactly one lane advances
  }
  if (lane < p.k) {
    if (p.topk_logprob) p.topk_logprob[(size_t)row * p.k + lane] = my_v - lse;
    if (p.topk_index) p.topk_index[(size_t)row * p.k + lane] = my_i;
  }
  if (lane == 0) {
    const int tgt = p.targets[row];
    const bool valid = (tgt >= 0) && (tgt < p.V);
    p.lse[row] = lse;
    p.target_logprob[row] = valid ? (p.zt[row] - lse) : 0.f;
    p.entropy[row] = (float)(lnS - U / S);
    p.conf[row] = lse - acc / (float)p.k;   // -(1/k) sum_j (z_(j) - lse)
  }
}

}  // namespace sq
