// sq_prepare_kernel.cuh -- SURVEY section 8(f)-2, the step before the path: gather the positions whose
// next-token distribution is wanted and apply the scorer's final RMSNorm,
//
//   H[t,:] = bf16( x / sqrt(mean_j x_j^2 + eps) * gain ),   x = X[pos[t],:]
//
// Token i of a trajectory is scored by log p(. | t_<i, Q) (Eq. 3), i.e. by the hidden state
// of the position before it, and only the |tau| trajectory tokens are averaged (Eq. 4): the
// caller's `pos` carries the shift and the packing, this kernel the gather and the normalisation.
//
// HBM-bound (2*d bytes read + 2*d bytes written per row), so it is NOT folded into kernel 1's TMA producer:
// that would put an elementwise pass over every A stage on the SM that runs the MMAs to save 0.3 % of the
// step.  One warp per row, rows grid-strided.  sq_prepare_reg_kernel<NV> (d <= 256*NV) loads the whole row into
// registers with NV independent 16-byte loads per lane, so HBM is touched once per byte and all of a row's loads
// are in flight together; sq_prepare_kernel is the general two-pass form (the second pass re-reads the row from
// L1/L2).  fp32 arithmetic, one rounding to bf16 (reading #20).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace sq {

constexpr int PREP_WARPS = 8;
constexpr int PREP_UNROLL = 4;   // 16-byte loads in flight per lane in pass 1

struct PrepareParams {
  const uint4* X;        // bf16 [N, d] viewed as 16-byte vectors
  const int32_t* pos;    // [T] rows of X, or null = identity (T rows, no gather)
  const uint4* gain;     // bf16 [d]
  uint4* H;              // bf16 [T, d]
  int T, N, d;
  float eps;
};

__device__ __forceinline__ void unpack8(const uint4& v, float (&f)[8]) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    f[2 * i] = __uint_as_float(w[i] << 16);            // bf16 -> fp32 is a 16-bit shift
    f[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
}
__device__ __forceinline__ uint32_t pack2(float lo, float hi) {
  const __nv_bfloat162 b = __floats2bfloat162_rn(lo, hi);   // round to nearest even
  return *reinterpret_cast<const uint32_t*>(&b);
}

__global__ void __launch_bounds__(PREP_WARPS * 32) sq_prepare_kernel(const PrepareParams p) {
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const int nvec = p.d >> 3;
  for (int t = blockIdx.x * PREP_WARPS + warp; t < p.T; t += gridDim.x * PREP_WARPS) {
    int src = p.pos ? __ldg(p.pos + t) : t;
    src = min(max(src, 0), p.N - 1);                   // contents are trusted; never read outside X
    const uint4* x = p.X + (size_t)src * nvec;
    float ss[PREP_UNROLL];
#pragma unroll
    for (int u = 0; u < PREP_UNROLL; ++u) ss[u] = 0.f;
    for (int v0 = 0; v0 < nvec; v0 += 32 * PREP_UNROLL) {
      uint4 q[PREP_UNROLL];
#pragma unroll
      for (int u = 0; u < PREP_UNROLL; ++u) {
        const int v = v0 + u * 32 + lane;
        q[u] = (v < nvec) ? x[v] : make_uint4(0u, 0u, 0u, 0u);
      }
#pragma unroll
      for (int u = 0; u < PREP_UNROLL; ++u) {
        float f[8];
        unpack8(q[u], f);
#pragma unroll
        for (int i = 0; i < 8; ++i) ss[u] = fmaf(f[i], f[i], ss[u]);
      }
    }
    float s = (ss[0] + ss[1]) + (ss[2] + ss[3]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    const float inv = 1.0f / sqrtf(s / (float)p.d + p.eps);
    uint4* h = p.H + (size_t)t * nvec;
    for (int v = lane; v < nvec; v += 32) {
      float f[8], g[8];
      unpack8(x[v], f);
      unpack8(__ldg(p.gain + v), g);
      uint4 o;
      o.x = pack2(f[0] * inv * g[0], f[1] * inv * g[1]);
      o.y = pack2(f[2] * inv * g[2], f[3] * inv * g[3]);
      o.z = pack2(f[4] * inv * g[4], f[5] * inv * g[5]);
      o.w = pack2(f[6] * inv * g[6], f[7] * inv * g[7]);
      h[v] = o;
    }
  }
}

// Register-resident form: lane l holds vectors l, l+32, ..., l+32*(NV-1) of the row.
constexpr int PREP_REG_WARPS = 4;   // 128-thread CTAs: at ~150 registers (NV = 16) three of them fit on an SM
template <int NV>
__global__ void __launch_bounds__(PREP_REG_WARPS * 32) sq_prepare_reg_kernel(const PrepareParams p) {
  extern __shared__ uint4 s_gain[];                    // the gain vector, staged once per (persistent) CTA
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const int nvec = p.d >> 3;
  for (int v = threadIdx.x; v < nvec; v += PREP_REG_WARPS * 32) s_gain[v] = __ldg(p.gain + v);
  __syncthreads();
  for (int t = blockIdx.x * PREP_REG_WARPS + warp; t < p.T; t += gridDim.x * PREP_REG_WARPS) {
    int src = p.pos ? __ldg(p.pos + t) : t;
    src = min(max(src, 0), p.N - 1);
    const uint4* x = p.X + (size_t)src * nvec;
    uint4 q[NV];
#pragma unroll
    for (int u = 0; u < NV; ++u) {
      const int v = u * 32 + lane;
      q[u] = (v < nvec) ? x[v] : make_uint4(0u, 0u, 0u, 0u);
    }
    float ss[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int u = 0; u < NV; ++u) {
      float f[8];
      unpack8(q[u], f);
#pragma unroll
      for (int i = 0; i < 8; ++i) ss[u & 3] = fmaf(f[i], f[i], ss[u & 3]);
    }
    float s = (ss[0] + ss[1]) + (ss[2] + ss[3]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    const float inv = 1.0f / sqrtf(s / (float)p.d + p.eps);
    uint4* h = p.H + (size_t)t * nvec;
#pragma unroll
    for (int u = 0; u < NV; ++u) {
      const int v = u * 32 + lane;
      if (v < nvec) {
        float f[8], g[8];
        unpack8(q[u], f);
        unpack8(s_gain[v], g);
        uint4 o;
        o.x = pack2(f[0] * inv * g[0], f[1] * inv * g[1]);
        o.y = pack2(f[2] * inv * g[2], f[3] * inv * g[3]);
        o.z = pack2(f[4] * inv * g[4], f[5] * inv * g[5]);
        o.w = pack2(f[6] * inv * g[6], f[7] * inv * g[7]);
        h[v] = o;
      }
    }
  }
}

}  // namespace sq
