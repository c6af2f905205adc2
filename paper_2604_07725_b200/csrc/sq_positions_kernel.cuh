// sq_positions_kernel.cuh -- the index arithmetic of the step before the path, on the device.
//
// A packed prefill holds, for candidate b, query_lens[b] query tokens followed by traj_lens[b] trajectory tokens.
// Token i (i = 1..|tau|) of a trajectory is scored by log p(. | t_<i, Q) (Eq. 3): by the hidden state of
// the packed row just before it; only the |tau| trajectory tokens are averaged (Eq. 4).  So
//     cu[b+1] = cu[b] + traj_lens[b],   base_b = sum_{c<b} (query_lens[c] + traj_lens[c]),
//     pos[cu[b] + i] = base_b + query_lens[b] - 1 + i.
// sq_positions_scan_kernel (one CTA) scans the B lengths; sq_positions_fill_kernel (one CTA per candidate) writes
// the rows.  Also here: the neutral element of the shard merge (sq_score_neutral_shard_state).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sq {

struct PositionsParams {
  const int32_t* query_lens;   // [B]
  const int32_t* traj_lens;    // [B]
  int B;
  int num_tokens;              // what the caller says sum traj_lens is
  int32_t* pos;                // [num_tokens]
  int32_t* cu;                 // [B + 1]
  int* base;                   // [B + 1] ctx scratch: packed start of every candidate
  int32_t* status;             // [1] or null
};

__global__ void __launch_bounds__(1024) sq_positions_scan_kernel(const PositionsParams p) {
  __shared__ long long warp_tok[32], warp_row[32];
  __shared__ int bad_total;
  if (threadIdx.x == 0) bad_total = 0;
  __syncthreads();
  // thread t owns the `per` consecutive candidates [t*per, (t+1)*per): one block scan of (tokens, packed rows)
  const int per = (p.B + 1023) / 1024;
  const int b_lo = min(p.B, (int)threadIdx.x * per), b_hi = min(p.B, b_lo + per);
  long long tok = 0, row = 0;
  int bad = 0;
  for (int b = b_lo; b < b_hi; ++b) {
    const int q = p.query_lens[b], n = p.traj_lens[b];
    bad += (q < 0 || n < 0 || (n > 0 && q < 1)) ? 1 : 0;
    tok += max(n, 0);
    row += max(q, 0) + max(n, 0);
  }
  long long xt = tok, xr = row;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const long long yt = __shfl_up_sync(0xffffffffu, xt, off), yr = __shfl_up_sync(0xffffffffu, xr, off);
    if (lane >= off) { xt += yt; xr += yr; }
  }
  if (lane == 31) { warp_tok[warp] = xt; warp_row[warp] = xr; }
  if (bad) atomicAdd(&bad_total, bad);
  __syncthreads();
  long long ot = 0, orow = 0;
  for (int w = 0; w < warp; ++w) { ot += warp_tok[w]; orow += warp_row[w]; }
  long long ct = ot + xt - tok, cr = orow + xr - row;   // exclusive prefixes of this thread's first candidate
  if (threadIdx.x == 0) p.cu[0] = 0;
  for (int b = b_lo; b < b_hi; ++b) {
    p.base[b] = (int)cr;
    ct += max(p.traj_lens[b], 0);
    cr += max(p.query_lens[b], 0) + max(p.traj_lens[b], 0);
    p.cu[b + 1] = (int)ct;
  }
  if (threadIdx.x == 1023 && p.status) {
    long long total = 0;
    for (int w = 0; w < 32; ++w) total += warp_tok[w];
    *p.status = bad_total + (total != (long long)p.num_tokens ? 1 : 0);
  }
}

__global__ void __launch_bounds__(256) sq_positions_fill_kernel(const PositionsParams p) {
  const int b = blockIdx.x;
  const int c0 = p.cu[b], c1 = min(p.cu[b + 1], p.num_tokens);   // never write past the caller's array
  const int first = p.base[b] + p.query_lens[b] - 1;             // the row that predicts trajectory token 1
  for (int t = c0 + (int)threadIdx.x; t < c1; t += 256) p.pos[t] = max(first + (t - c0), 0);
}

// m[T] s[T] u[T] cs[T] cu[T] topv[cap][T] topi[cap][T] zt[T]: the packed state of a shard without vocabulary rows
__global__ void __launch_bounds__(256) sq_neutral_state_kernel(float* st, int T, int cap) {
  const long long words = (6LL + 2LL * cap) * T;
  for (long long w = (long long)blockIdx.x * 256 + threadIdx.x; w < words; w += (long long)gridDim.x * 256) {
    const long long sec = w / T;   // which array of the layout
    float v = 0.f;                 // s, u, cs, cu, zt
    if (sec == 0 || (sec >= 5 && sec < 5 + cap)) v = -1.0e30f;             // m and the list values: "nothing seen"
    else if (sec >= 5 + cap && sec < 5 + 2LL * cap) v = __int_as_float(-1);  // list ids: empty slot
    st[w] = v;
  }
}

}  // namespace sq
