// sq_finalize_kernel.cuh -- step a6: merge the vocab-chunk partial states of every row and finalise.
//
//   lse = M + ln S,  M = max_c m_c,  S = sum_c s_c e^{m_c - M}      (merged in fp64)
//   entropy = ln S - U / S,  U = sum_c e^{m_c - M} (u_c + (m_c - M) s_c)
//   target_logprob = z_target - lse
//   topk_logprob_j = z_(j) - lse,  conf = c(i) = -(1/k) sum_j topk_logprob_j    (Eq. 3)
//
// One warp per token row; lane c holds the state of chunks c, c+32, ... (num_chunks <= 160).  The running max / sum /
// entropy merge is a warp-shuffle reduction; the top-k merge is k rounds of a warp arg-max over the
// heads of the per-chunk sorted lists (ties: larger value first, then smaller vocabulary id).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sq {

struct FinalizeParams {
  int T, V, k, cap, num_chunks;
  // Partial states may come from several vocab-parallel shards ("ranks"): chunk c lives in rank c / chunks_per_rank,
  // whose arrays start rank_stride 4-byte words after the previous rank's (one packed state buffer per rank, gathered
  // back to back).  One rank: chunks_per_rank = num_chunks, rank_stride = 0.
  int chunks_per_rank;
  long long rank_stride;
  int num_ranks;
  int vstart[33];           // ranks > 1: rank r owns vocabulary ids [vstart[r], vstart[r+1]) -- whose zt is the target's
  int vocab_offset;         // EMIT mode: this shard's columns are global ids [vocab_offset, vocab_offset + V)
  // EMIT mode (sq_score_run_shard): instead of finalising, write the merged state as ONE chunk in the same format
  float* out_m; float* out_s; float* out_u; float* out_cs; float* out_cu;   // [T]
  float* out_topv; int32_t* out_topi;                                        // [cap][T]
  float* out_zt;                                                             // [T]
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
constexpr int FIN_MAX_NL = 5;                      // lists per lane
constexpr int FIN_MAX_CHUNKS = 32 * FIN_MAX_NL;    // 160 vocab chunks per row at most

// NL = lists (vocab chunks) per lane: 1 for the prefill-shaped plans (num_chunks <= 32), FIN_MAX_NL otherwise.
// EMIT = write the merged state of this shard (m, s, u with their residues, k-entry list, target logit) for the
// vocab-parallel exchange instead of the final per-token outputs.
// LPR = lanes per row: 32 (one warp per row), or 8 when there are at most 8 chunks (the large prefill plans: 6), so
// that a warp merges four rows at once and the k rounds of arg-max shuffles are shared by four times as many rows.
template <int NL, bool EMIT, int LPR = 32>
__global__ void __launch_bounds__(FIN_WARPS * 32)
sq_finalize_kernel(const FinalizeParams p) {
  static_assert(LPR == 32 || (LPR == 8 && NL == 1), "8 lanes per row needs one list per lane");
  cudaGridDependencySynchronize();   // launched with programmatic serialization behind kernel 1 (or stand-alone: no-op)
  constexpr int RPW = 32 / LPR;      // rows per warp
  const int lane = (threadIdx.x & 31) % LPR;   // position inside the row's lane group = chunk index (+ 32 i)
  const int row_raw = (blockIdx.x * FIN_WARPS + (threadIdx.x >> 5)) * RPW + (threadIdx.x & 31) / LPR;
  if ((blockIdx.x * FIN_WARPS + (threadIdx.x >> 5)) * RPW >= p.T) return;   // the whole warp is past the end
  const bool live = row_raw < p.T;   // lanes of a dead row still take part in the shuffles, on row T-1's data
  const int row = live ? row_raw : p.T - 1;
  const unsigned FULL = 0xffffffffu;
  const float NEG = -1.0e30f;
  // lane owns chunks lane, lane + 32, ... (one per lane in the prefill-shaped plans, up to
  // NL in the decode-shaped ones where every SM sweeps its own slice of the vocabulary)
  size_t base1[NL], basek[NL];   // word offsets of this lane's chunks: scalar arrays / first list entry
#pragma unroll
  for (int i = 0; i < NL; ++i) {
    const int c = lane + 32 * i;
    const int r = c / p.chunks_per_rank, cl = c - r * p.chunks_per_rank;
    base1[i] = (size_t)r * p.rank_stride + (size_t)cl * p.T + row;
    basek[i] = (size_t)r * p.rank_stride + (size_t)cl * p.cap * p.T + row;
  }
  float M = NEG;
#pragma unroll
  for (int i = 0; i < NL; ++i) {
    const int c = lane + 32 * i;
    if (c < p.num_chunks) M = fmaxf(M, p.part_m[base1[i]]);
  }
#pragma unroll
  for (int off = LPR / 2; off > 0; off >>= 1) M = fmaxf(M, __shfl_xor_sync(FULL, M, off));
  // the merge runs in fp64: S - 1 of a peaked row is ~1e-4 and carries the whole entropy
  double S = 0.0, U = 0.0;
#pragma unroll
  for (int i = 0; i < NL; ++i) {
    const int c = lane + 32 * i;
    if (c < p.num_chunks) {
      const size_t o = base1[i];
      const double s_c = (double)p.part_s[o] - (double)p.part_cs[o];
      const double u_c = (double)p.part_u[o] - (double)p.part_cu[o];
      const double dm = (double)p.part_m[o] - (double)M;
      const double w = exp(dm);
      S += w * s_c;
      U += w * (u_c + dm * s_c);
    }
  }
#pragma unroll
  for (int off = LPR / 2; off > 0; off >>= 1) {
    S += __shfl_xor_sync(FULL, S, off);
    U += __shfl_xor_sync(FULL, U, off);
  }
  const double lnS = log(S);
  const float lse = (float)((double)M + lnS);

  // ---- top-k merge: the lane walks its chunks' descending lists; hv/hi[i] = head of list i, nv/ni[i] = the entry
  // behind it, loaded one pop ahead so that its latency hides behind the next round's shuffles
  int pos[NL];
  float hv[NL], nv[NL];
  int hi[NL], ni[NL];
  auto load_at = [&](int i, int at, float& v, int& id) -> void {
    const int c = lane + 32 * i;
    v = NEG; id = 0x7fffffff;
    if (c < p.num_chunks && at < p.cap) {
      const size_t oj = basek[i] + (size_t)at * p.T;
      v = p.part_topv[oj];
      id = p.part_topi[oj];
      if (id < 0) { v = NEG; id = 0x7fffffff; }   // unfilled slot
    }
  };
#pragma unroll
  for (int i = 0; i < NL; ++i) { pos[i] = 0; load_at(i, 0, hv[i], hi[i]); load_at(i, 1, nv[i], ni[i]); }
  float acc = 0.f;       // sum of the k best logits
  float my_v = 0.f; int my_i = 0;   // lane j keeps the j-th winner for a coalesced store
  for (int j = 0; j < p.k; ++j) {
    float lv = hv[0]; int li = hi[0];
#pragma unroll
    for (int i = 1; i < NL; ++i)
      if (hv[i] > lv || (hv[i] == lv && hi[i] < li)) { lv = hv[i]; li = hi[i]; }
    float bv = lv; int bi = li;
#pragma unroll
    for (int off = LPR / 2; off > 0; off >>= 1) {
      const float ov = __shfl_xor_sync(FULL, bv, off);
      const int oi = __shfl_xor_sync(FULL, bi, off);
      if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    acc += bv;
    if constexpr (LPR == 32) {
      if (lane == j) { my_v = bv; my_i = bi; }
    } else if (lane == (j & (LPR - 1)) && live) {   // too few lanes to park k winners: store the j-th right away
      if (EMIT) {
        p.out_topv[(size_t)j * p.T + row] = bv;
        p.out_topi[(size_t)j * p.T + row] = bv > NEG ? bi : -1;
      } else {
        if (p.topk_logprob) p.topk_logprob[(size_t)row * p.k + j] = bv - lse;
        if (p.topk_index) p.topk_index[(size_t)row * p.k + j] = bi;
      }
    }
    if (li == bi && lv == bv) {   // vocabulary ids are unique: exactly one list of one lane advances
#pragma unroll
      for (int i = 0; i < NL; ++i)
        if (hi[i] == bi && hv[i] == bv) { ++pos[i]; hv[i] = nv[i]; hi[i] = ni[i]; load_at(i, pos[i] + 1, nv[i], ni[i]); }
    }
  }
  if (EMIT) {
    // the shard's merged state, one chunk: s and u keep their fp64 precision as value + residue (true = s - cs)
    if constexpr (LPR == 32) {
      if (lane < p.cap) {
        p.out_topv[(size_t)lane * p.T + row] = lane < p.k ? my_v : NEG;
        p.out_topi[(size_t)lane * p.T + row] = (lane < p.k && my_v > NEG) ? my_i : -1;
      }
    } else if (live) {
      for (int j = p.k + lane; j < p.cap; j += LPR) {   // the list slots past k are empty
        p.out_topv[(size_t)j * p.T + row] = NEG;
        p.out_topi[(size_t)j * p.T + row] = -1;
      }
    }
    if (lane == 0 && live) {
      const float s_hi = (float)S, u_hi = (float)U;
      p.out_m[row] = M;
      p.out_s[row] = s_hi; p.out_cs[row] = (float)((double)s_hi - S);
      p.out_u[row] = u_hi; p.out_cu[row] = (float)((double)u_hi - U);
      // the target's logit exists only on the shard that owns its column (kernel 1 writes zt[row] only there)
      const int tl = p.targets[row] - p.vocab_offset;
      p.out_zt[row] = (tl >= 0 && tl < p.V) ? p.zt[row] : 0.f;
    }
    return;
  }
  if constexpr (LPR == 32) {
    if (lane < p.k) {
      if (p.topk_logprob) p.topk_logprob[(size_t)row * p.k + lane] = my_v - lse;
      if (p.topk_index) p.topk_index[(size_t)row * p.k + lane] = my_i;
    }
  }
  if (lane == 0 && live) {
    const int tgt = p.targets[row];
    const bool valid = (tgt >= 0) && (tgt < p.V);
    size_t zo = row;
    if (p.num_ranks > 1 && valid) {
      int r = 0;
      while (r + 1 < p.num_ranks && tgt >= p.vstart[r + 1]) ++r;
      zo += (size_t)r * p.rank_stride;
    }
    p.lse[row] = lse;
    p.target_logprob[row] = valid ? (p.zt[zo] - lse) : 0.f;
    p.entropy[row] = (float)(lnS - U / S);
    p.conf[row] = lse - acc / (float)p.k;   // -(1/k) sum_j (z_(j) - lse)
  }
}

}  // namespace sq
