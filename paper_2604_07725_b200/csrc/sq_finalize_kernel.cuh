// sq_finalize_kernel.cuh -- step a6: merge the vocab-chunk partial states of every row and finalise.
//
//   lse = M + ln S,  M = max_c m_c,  S = sum_c s_c e^{m_c - M}      (merged in fp64)
//   entropy = ln S - U / S,  U = sum_c e^{m_c - M} (u_c + (m_c - M) s_c)
//   target_logprob = z_target - lse
//   topk_logprob_j = z_(j) - lse,  conf = c(i) = -(1/k) sum_j topk_logprob_j    (Eq. 3)
//
// One warp per token row; lane c holds the state of chunk c (num_chunks <= 32; wider rows: sq_finalize_wide_kernel).  The running max / sum /
// entropy merge is a warp-shuffle reduction; the top-k merge is k rounds of a warp arg-max over the
// heads of the per-chunk sorted lists (ties: larger value first, then smaller vocabulary id).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sq {

struct FinalizeParams {
  int T, V, k, cap, num_chunks;
  // Partial states may come from several vocab-parallel shards ("ranks"): chunk c lives in rank c / chunks_per_rank,
  // whose arrays start rank_off[r] 4-byte words after rank 0's: r * (words of a packed state) when the states were
  // gathered back to back (sq_score_merge_shards), or the distance between two buffers anywhere in the unified address
  // space -- the peers' own state buffers, read in place over NVLink (sq_score_merge_shards_peer).  One rank:
  // chunks_per_rank = num_chunks, rank_off[0] = 0.
  int chunks_per_rank;
  int num_ranks;
  long long rank_off[32];
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
  // Small runs (T <= FIN_TAIL_MAX_T, decode-shaped): kernel 2's work is a few hundred tokens, i.e. pure launch latency
  // as a kernel of its own, so the LAST CTA of this grid to finish does it (step a7; same definitions as
  // sq_reduce_kernel.cuh).  tail_B = 0: no tail (kernel 2 follows as a launch).
  int tail_B, tail_window;
  const int32_t* tail_cu;   // [B+1]
  float* tail_out_lp; float* tail_out_ent; float* tail_out_conf; float* tail_out_min;   // [B]
  unsigned int* tail_counter;   // ctx-owned, zero between runs
};

constexpr int FIN_WARPS = 8;
constexpr int FIN_TAIL_MAX_T = 256;                // largest T whose per-sequence reductions run in the finalize kernel's tail

// Step a7 for a small run, by one CTA, from the per-token outputs the grid has just written (sq_reduce_kernel.cuh states
// the definitions): per sequence the mean target log-prob over valid targets, mean entropy, C(tau) = mean c(i) (Eq. 4,
// PAPER.md:160) and the minimum over stride-1 full windows of length w' = min(w, L) of the window mean of c(i); an
// empty sequence gives NaNs.  One warp per sequence; fp64 sums and an fp64 prefix of c(i) (L <= 256), so every window
// sum is exact to fp64 rounding.
template <int NWARPS>
__device__ __forceinline__ void fin_tail_reduce(const FinalizeParams& p, double* s_prefix) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* pre = s_prefix + warp * (FIN_TAIL_MAX_T + 1);
  for (int b = warp; b < p.tail_B; b += NWARPS) {
    // cu_seqlens is device data nobody has checked (sq_score_positions emits an inconsistent one when its status is
    // non-zero): clamped into [0, T], T <= FIN_TAIL_MAX_T, so that `pre` and the per-token arrays are never overrun
    const int s0 = min(max(p.tail_cu[b], 0), p.T), s1 = min(max(p.tail_cu[b + 1], s0), p.T);
    const int L = s1 - s0;
    if (L <= 0) {
      if (lane == 0) { const float nan = __int_as_float(0x7fc00000); p.tail_out_lp[b] = nan; p.tail_out_ent[b] = nan; p.tail_out_conf[b] = nan; p.tail_out_min[b] = nan; }
      continue;
    }
    double a_lp = 0.0, a_n = 0.0, a_en = 0.0;
    for (int i = lane; i < L; i += 32) {
      const int t = s0 + i;
      const bool valid = (unsigned)p.targets[t] < (unsigned)p.V;
      a_lp += valid ? (double)__ldcg(p.target_logprob + t) : 0.0;
      a_n += valid ? 1.0 : 0.0;
      a_en += (double)__ldcg(p.entropy + t);
    }
    // inclusive fp64 prefix of c(i): 32 tokens per pass, warp scan + carry
    double carry = 0.0;
    if (lane == 0) pre[0] = 0.0;
    for (int i0 = 0; i0 < L; i0 += 32) {
      const int i = i0 + lane;
      double x = i < L ? (double)__ldcg(p.conf + s0 + i) : 0.0;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const double y = __shfl_up_sync(0xffffffffu, x, off);
        if (lane >= off) x += y;
      }
      if (i < L) pre[i + 1] = carry + x;
      carry += __shfl_sync(0xffffffffu, x, 31);
    }
    __syncwarp();
    const int w = min(p.tail_window, L);
    double best = 1.0e300;
    for (int j = lane; j + w <= L; j += 32) best = fmin(best, pre[j + w] - pre[j]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      a_lp += __shfl_xor_sync(0xffffffffu, a_lp, off);
      a_n += __shfl_xor_sync(0xffffffffu, a_n, off);
      a_en += __shfl_xor_sync(0xffffffffu, a_en, off);
      best = fmin(best, __shfl_xor_sync(0xffffffffu, best, off));
    }
    if (lane == 0) {
      p.tail_out_lp[b] = a_n > 0.0 ? (float)(a_lp / a_n) : __int_as_float(0x7fc00000);
      p.tail_out_ent[b] = (float)(a_en / (double)L);
      p.tail_out_conf[b] = (float)(carry / (double)L);
      p.tail_out_min[b] = (float)(best / (double)w);
    }
    __syncwarp();                                  // `pre` is reused by the warp's next sequence
  }
}
constexpr int FIN_MAX_CHUNKS = 160;                // vocab chunks per row at most

// NL = lists (vocab chunks) per lane: 1 (at most 32 chunks per row; more take sq_finalize_wide_kernel below).
// EMIT = write the merged state of this shard (m, s, u with their residues, k-entry list, target logit) for the
// vocab-parallel exchange instead of the final per-token outputs.
// LPR = lanes per row: 32 (one warp per row), or 8 when there are at most 8 chunks (the large prefill plans: 6), so
// that a warp merges four rows at once and the k rounds of arg-max shuffles are shared by four times as many rows.
template <int NL, bool EMIT, int LPR>
__device__ __forceinline__ void fin_merge_rows(const FinalizeParams& p) {
  static_assert(LPR == 32 || (LPR == 8 && NL == 1), "8 lanes per row needs one list per lane");
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
  long long base1[NL], basek[NL];   // word offsets of this lane's chunks (signed: a peer's buffer may lie below rank 0's)
#pragma unroll
  for (int i = 0; i < NL; ++i) {
    const int c = lane + 32 * i;
    const int r = c / p.chunks_per_rank, cl = c - r * p.chunks_per_rank;
    base1[i] = (long long)p.rank_off[r & 31] + (long long)cl * p.T + row;
    basek[i] = (long long)p.rank_off[r & 31] + (long long)cl * p.cap * p.T + row;
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
      const long long o = base1[i];
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
  float hv[NL] = {}, nv[NL] = {};
  int hi[NL] = {}, ni[NL] = {};
  // raw load of list entry `at` (id < 0 = unfilled slot / past the end); the id is NOT examined here, so that the load
  // issued at a pop is a true prefetch: nothing waits for it until the entry becomes a head, one pop of the same list later
  auto load_at = [&](int i, int at, float& v, int& id) -> void {
    const int c = lane + 32 * i;
    v = NEG; id = -1;
    if (c < p.num_chunks && at < p.cap) {
      const long long oj = basek[i] + (long long)at * p.T;
      v = p.part_topv[oj];
      id = p.part_topi[oj];
    }
  };
  auto promote = [&](int i) -> void {              // the prefetched entry becomes the head
    const bool empty = ni[i] < 0;
    hv[i] = empty ? NEG : nv[i];
    hi[i] = empty ? 0x7fffffff : ni[i];
  };
#pragma unroll
  for (int i = 0; i < NL; ++i) { pos[i] = 0; load_at(i, 0, nv[i], ni[i]); promote(i); load_at(i, 1, nv[i], ni[i]); }
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
        if (hi[i] == bi && hv[i] == bv) { ++pos[i]; promote(i); load_at(i, pos[i] + 1, nv[i], ni[i]); }
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
    long long zo = row;
    if (p.num_ranks > 1 && valid) {
      int r = 0;
      while (r + 1 < p.num_ranks && tgt >= p.vstart[r + 1]) ++r;
      zo += p.rank_off[r];
    }
    p.lse[row] = lse;
    p.target_logprob[row] = valid ? (p.zt[zo] - lse) : 0.f;
    p.entropy[row] = (float)(lnS - U / S);
    p.conf[row] = lse - acc / (float)p.k;   // -(1/k) sum_j (z_(j) - lse)
  }
}

template <int NL, bool EMIT, int LPR = 32>
__global__ void __launch_bounds__(FIN_WARPS * 32)
sq_finalize_kernel(const FinalizeParams p) {
  cudaGridDependencySynchronize();   // launched with programmatic serialization behind kernel 1 (or stand-alone: no-op)
  fin_merge_rows<NL, EMIT, LPR>(p);
  if constexpr (!EMIT) {
    if (p.tail_B > 0) {              // grid-uniform: a small run, the last CTA to finish does kernel 2's work
      __shared__ double s_prefix[FIN_WARPS * (FIN_TAIL_MAX_T + 1)];
      __shared__ int s_is_last;
      __threadfence();               // this thread's per-token outputs are visible before the CTA is counted
      __syncthreads();
      if (threadIdx.x == 0) s_is_last = (atomicAdd(p.tail_counter, 1u) == gridDim.x - 1) ? 1 : 0;
      __syncthreads();
      if (s_is_last) {
        __threadfence();
        fin_tail_reduce<FIN_WARPS>(p, s_prefix);
        if (threadIdx.x == 0) *p.tail_counter = 0u;   // zero again for the next run
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------------
// Wide form, for rows swept by MORE than 32 vocab chunks (decode-shaped plans: every SM streams its own stripe of W, up
// to 160 chunks per row; few rows).  One CTA of FIN_WIDE_WARPS warps per row, thread c = chunk c.  The statistics are
// one block reduction.  The top-k merge has NO serial rounds (k rounds of warp arg-max cost 20-35 us for 64 rows, all of
// it dependent-instruction latency); it is a selection by counting:
//   1. every thread loads its chunk's whole sorted list (CAP independent loads);
//   2. x = the k-th largest of the C list HEADS (rank by counting over shared memory).  k lists hold an entry >= x, so
//      x bounds the row's k-th best from below and only entries >= x can be among the k best: a few dozen of C * CAP;
//   3. the survivors are compacted into shared memory (block prefix sum of the per-list counts; a list is sorted, so
//      its survivors are a prefix) and ranked by counting against one another (value desc, id asc): the survivor of
//      rank j < k IS the j-th best, and writes itself to slot j.
// 23.9 us (one warp per row, 5 lists per lane) -> 21.7 us (two levels of warp arg-max rounds) -> this form.
constexpr int FIN_WIDE_WARPS = FIN_MAX_CHUNKS / 32;   // 5
constexpr int FIN_WIDE_THREADS = FIN_WIDE_WARPS * 32;
constexpr int FIN_WIDE_CAND = 1024;                   // k lists of CAP entries at most survive: 32 * 32

template <int CAP, bool EMIT>
__global__ void __launch_bounds__(FIN_WIDE_THREADS)
sq_finalize_wide_kernel(const FinalizeParams p) {
  __shared__ float s_max[FIN_WIDE_WARPS];
  __shared__ double s_S[FIN_WIDE_WARPS], s_U[FIN_WIDE_WARPS];
  __shared__ float s_head[FIN_WIDE_THREADS];
  __shared__ int s_cnt[FIN_WIDE_WARPS];
  __shared__ float s_thr;
  __shared__ float s_cv[FIN_WIDE_CAND];
  __shared__ int s_ci[FIN_WIDE_CAND];
  __shared__ float s_win[32];
  __shared__ int s_is_last;
  cudaGridDependencySynchronize();
  const int row = blockIdx.x;                       // grid = T rows
  const int c = threadIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned FULL = 0xffffffffu;
  const float NEG = -1.0e30f, EMPTY = -1.0e20f;     // list values below EMPTY are unfilled slots (no logit is that small)
  const bool has = c < p.num_chunks;
  const int r = has ? c / p.chunks_per_rank : 0, cl = has ? c - r * p.chunks_per_rank : 0;
  const long long base1 = p.rank_off[r & 31] + (long long)cl * p.T + row;
  const long long basek = p.rank_off[r & 31] + (long long)cl * p.cap * p.T + row;
  // ---- every load this thread needs, issued together: the chunk's statistics and its whole list of values
  float m_c = NEG, s_c = 0.f, cs_c = 0.f, u_c = 0.f, cu_c = 0.f;
  float lv[CAP];
#pragma unroll
  for (int j = 0; j < CAP; ++j) lv[j] = NEG;
  if (has) {
    m_c = p.part_m[base1]; s_c = p.part_s[base1]; cs_c = p.part_cs[base1]; u_c = p.part_u[base1]; cu_c = p.part_cu[base1];
#pragma unroll
    for (int j = 0; j < CAP; ++j) lv[j] = p.part_topv[basek + (long long)j * p.T];
  }
  float M = m_c;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) M = fmaxf(M, __shfl_xor_sync(FULL, M, off));
  if (lane == 0) s_max[warp] = M;
  const float head = lv[0] > EMPTY ? lv[0] : NEG;
  s_head[c] = head;
  __syncthreads();
  M = s_max[0];
#pragma unroll
  for (int w = 1; w < FIN_WIDE_WARPS; ++w) M = fmaxf(M, s_max[w]);
  double S = 0.0, U = 0.0;                          // fp64: S - 1 of a peaked row carries the whole entropy
  if (has) {
    const double sc = (double)s_c - (double)cs_c, uc = (double)u_c - (double)cu_c;
    const double dm = (double)m_c - (double)M;
    const double w = exp(dm);
    S = w * sc;
    U = w * (uc + dm * sc);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    S += __shfl_xor_sync(FULL, S, off);
    U += __shfl_xor_sync(FULL, U, off);
  }
  if (lane == 0) { s_S[warp] = S; s_U[warp] = U; }
  // ---- 2. the k-th largest head, by counting (ties: the smaller chunk index ranks first, so ranks are distinct)
  int rank = 0;
#pragma unroll 8
  for (int q = 0; q < FIN_WIDE_THREADS; ++q) {
    const float h = s_head[q];
    rank += (h > head || (h == head && q < c)) ? 1 : 0;
  }
  if (rank == p.k - 1) s_thr = head;                // exactly one thread (k <= 32 < C non-empty lists)
  __syncthreads();
  const float thr = fmaxf(s_thr, EMPTY);
  // ---- 3. survivors: a prefix of every sorted list.  Entries ABOVE x come first in the buffer (at most k - 1 lists hold
  // any: they always fit); entries EQUAL to x follow and may be cut off when degenerate inputs tie by the thousand --
  // any of them is a correct k-th best, so the ones that fit are as good as the ones that do not.
  int cnt_gt = 0, cnt_ge = 0;
#pragma unroll
  for (int j = 0; j < CAP; ++j) { cnt_gt += (lv[j] > thr) ? 1 : 0; cnt_ge += (lv[j] >= thr) ? 1 : 0; }
  int inc = (cnt_gt << 16) | (cnt_ge - cnt_gt);     // both prefix sums in one scan (each below 2^15)
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int y = __shfl_up_sync(FULL, inc, off);
    if (lane >= off) inc += y;
  }
  if (lane == 31) s_cnt[warp] = inc;
  __syncthreads();
  int bs = inc - ((cnt_gt << 16) | (cnt_ge - cnt_gt)), tot = 0;
#pragma unroll
  for (int w = 0; w < FIN_WIDE_WARPS; ++w) { bs += (w < warp) ? s_cnt[w] : 0; tot += s_cnt[w]; }
  const int total_gt = tot >> 16, total = min(total_gt + (tot & 0xffff), FIN_WIDE_CAND);
  const int base_gt = bs >> 16, base_eq = total_gt + (bs & 0xffff);
#pragma unroll
  for (int j = 0; j < CAP; ++j) {
    const int at = j < cnt_gt ? base_gt + j : base_eq + (j - cnt_gt);
    if (j < cnt_ge && at < FIN_WIDE_CAND) {
      s_cv[at] = lv[j];
      s_ci[at] = p.part_topi[basek + (long long)j * p.T];
    }
  }
  if (c < 32) s_win[c] = NEG;
  __syncthreads();
  // ---- rank the survivors against one another; rank j < k is the j-th best (value desc, id asc; ids are unique)
  for (int t = c; t < total; t += FIN_WIDE_THREADS) {
    const float v = s_cv[t];
    const int id = s_ci[t];
    int rk = 0;
    for (int q = 0; q < total; ++q) {
      const float ov = s_cv[q];
      rk += (ov > v || (ov == v && s_ci[q] < id)) ? 1 : 0;
    }
    if (rk < p.k) {
      s_win[rk] = v;
      if (EMIT) {
        p.out_topv[(size_t)rk * p.T + row] = v;
        p.out_topi[(size_t)rk * p.T + row] = id;
      } else {
        if (p.topk_index) p.topk_index[(size_t)row * p.k + rk] = id;
      }
    }
  }
  __syncthreads();
  if (warp == 0) {
    S = 0.0; U = 0.0;
#pragma unroll
    for (int w = 0; w < FIN_WIDE_WARPS; ++w) { S += s_S[w]; U += s_U[w]; }   // fixed order
    const double lnS = log(S);
    const float lse = (float)((double)M + lnS);
    if (EMIT) {
      if (lane < p.cap && (lane >= p.k || s_win[lane] <= EMPTY)) {   // slots past k, and slots no entry filled
        p.out_topv[(size_t)lane * p.T + row] = NEG;
        p.out_topi[(size_t)lane * p.T + row] = -1;
      }
      if (lane == 0) {
        const float s_hi = (float)S, u_hi = (float)U;
        p.out_m[row] = M;
        p.out_s[row] = s_hi; p.out_cs[row] = (float)((double)s_hi - S);
        p.out_u[row] = u_hi; p.out_cu[row] = (float)((double)u_hi - U);
        const int tl = p.targets[row] - p.vocab_offset;
        p.out_zt[row] = (tl >= 0 && tl < p.V) ? p.zt[row] : 0.f;
      }
    } else {
      if (lane < p.k) {
        if (p.topk_logprob) p.topk_logprob[(size_t)row * p.k + lane] = s_win[lane] - lse;
        if (p.topk_index && s_win[lane] <= EMPTY) p.topk_index[(size_t)row * p.k + lane] = 0x7fffffff;   // fewer than k logits
      }
      if (lane == 0) {
        float acc = 0.f;
        for (int j = 0; j < p.k; ++j) acc += s_win[j];   // fixed order: deterministic
        const int tgt = p.targets[row];
        const bool valid = (tgt >= 0) && (tgt < p.V);
        p.lse[row] = lse;
        p.target_logprob[row] = valid ? (p.zt[row] - lse) : 0.f;   // the wide form serves single-rank runs only
        p.entropy[row] = (float)(lnS - U / S);
        p.conf[row] = lse - acc / (float)p.k;
      }
    }
  }
  // ---- small runs: the last CTA to finish does kernel 2's work
  if constexpr (!EMIT) {
    if (p.tail_B > 0) {
      __threadfence();
      __syncthreads();
      if (threadIdx.x == 0) s_is_last = (atomicAdd(p.tail_counter, 1u) == gridDim.x - 1) ? 1 : 0;
      __syncthreads();
      if (s_is_last) {
        __threadfence();
        __shared__ double s_prefix[FIN_WIDE_WARPS * (FIN_TAIL_MAX_T + 1)];
        fin_tail_reduce<FIN_WIDE_WARPS>(p, s_prefix);
        if (threadIdx.x == 0) *p.tail_counter = 0u;
      }
    }
  }
}

}  // namespace sq
