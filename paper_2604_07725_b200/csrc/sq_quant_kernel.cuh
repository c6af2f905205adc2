// sq_quant_kernel.cuh -- e4m3 quantisation for the FP8 variant of the scoring pass.
//
//   q[r, j] = e4m3_rn_sat( x[r, j] * (448 / amax) ),   scale = amax / 448,   x ~= q * scale
//
// amax is taken per row (H: one scale per token, applied for free in kernel 1's epilogue) or over the whole tensor
// (W: one scale for the LM head, so that no per-column multiply is needed per logit).  fp32 arithmetic: inv = 448 / amax
// and y = x * inv are one rounding each, so y is within 2 * 2^-24 of the exact x * 448 / amax; the parity test demands
// a correct e4m3 rounding of a value that close to the fp64 definition, and the fp64-decided code itself except at
// values that sit that close to a rounding boundary.  amax == 0 gives scale 1 and all-zero codes.  HBM-bound: 2 B read + 1 B
// written per element (per-tensor mode reads the tensor twice: amax pass, then quantise).
#pragma once
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace sq {

constexpr int QUANT_WARPS = 8;
constexpr float E4M3_MAX = 448.0f;

struct QuantParams {
  const uint4* X;        // bf16 [rows, d] as 16-byte vectors (8 elements)
  uint2* Q;              // e4m3 [rows, d] as 8-byte vectors (8 elements)
  float* scale;          // per-row: [rows] written; per-tensor: [1] written by sq_quant_scale_kernel, read here
  unsigned int* amax_bits;   // per-tensor: running max of |x| as fp32 bits (non-negative floats order like uints)
  long long rows;
  int d;
  int per_tensor;
};

__device__ __forceinline__ void q_unpack8(const uint4& v, float (&f)[8]) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    f[2 * i] = __uint_as_float(w[i] << 16);
    f[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
}
__device__ __forceinline__ float q_amax8(const uint4& v) {
  float f[8];
  q_unpack8(v, f);
  float m = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) m = fmaxf(m, fabsf(f[i]));
  return m;
}
__device__ __forceinline__ uint32_t q_code(float x, float inv) {
  const float y = fminf(fmaxf(__fmul_rn(x, inv), -E4M3_MAX), E4M3_MAX);
  return (uint32_t)__nv_cvt_float_to_fp8(y, __NV_SATFINITE, __NV_E4M3);
}
__device__ __forceinline__ uint2 q_pack8(const uint4& v, float inv) {
  float f[8];
  q_unpack8(v, f);
  uint2 o;
  o.x = q_code(f[0], inv) | (q_code(f[1], inv) << 8) | (q_code(f[2], inv) << 16) | (q_code(f[3], inv) << 24);
  o.y = q_code(f[4], inv) | (q_code(f[5], inv) << 8) | (q_code(f[6], inv) << 16) | (q_code(f[7], inv) << 24);
  return o;
}

// per-tensor pass 1: amax over everything
__global__ void __launch_bounds__(256) sq_quant_amax_kernel(const QuantParams p) {
  const long long nvec = p.rows * (p.d >> 3);
  float m = 0.f;
  for (long long v = (long long)blockIdx.x * 256 + threadIdx.x; v < nvec; v += (long long)gridDim.x * 256) m = fmaxf(m, q_amax8(p.X[v]));
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, off));
  if ((threadIdx.x & 31) == 0) atomicMax(p.amax_bits, __float_as_uint(m));
}
// per-tensor pass 1b: the scale from the amax
__global__ void sq_quant_scale_kernel(const QuantParams p) {
  const float amax = __uint_as_float(*p.amax_bits);
  p.scale[0] = amax > 0.f ? __fdiv_rn(amax, E4M3_MAX) : 1.f;
}

// quantise: one warp per row (per-row mode computes the row's amax first; the row is re-read from L1/L2)
__global__ void __launch_bounds__(QUANT_WARPS * 32) sq_quant_rows_kernel(const QuantParams p) {
  const int lane = threadIdx.x & 31;
  const int nvec = p.d >> 3;
  float amax_t = 0.f;
  if (p.per_tensor) amax_t = __uint_as_float(*p.amax_bits);
  for (long long r = (long long)blockIdx.x * QUANT_WARPS + (threadIdx.x >> 5); r < p.rows; r += (long long)gridDim.x * QUANT_WARPS) {
    const uint4* x = p.X + r * nvec;
    float amax = amax_t;
    if (!p.per_tensor) {
      amax = 0.f;
      for (int v = lane; v < nvec; v += 32) amax = fmaxf(amax, q_amax8(x[v]));
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, off));
      if (lane == 0) p.scale[r] = amax > 0.f ? __fdiv_rn(amax, E4M3_MAX) : 1.f;
    }
    const float inv = amax > 0.f ? __fdiv_rn(E4M3_MAX, amax) : 1.f;
    uint2* q = p.Q + r * nvec;
    for (int v = lane; v < nvec; v += 32) q[v] = q_pack8(x[v], inv);
  }
}

// Register-resident form (d <= 256 * NV): the row's NV 16-byte vectors per lane are loaded together, so the row is read
// from HBM once and all its loads are in flight at the same time (the pattern that took sq_prepare to 96 % of the copy peak).
constexpr int QUANT_REG_WARPS = 4;
template <int NV>
__global__ void __launch_bounds__(QUANT_REG_WARPS * 32) sq_quant_rows_reg_kernel(const QuantParams p) {
  const int lane = threadIdx.x & 31;
  const int nvec = p.d >> 3;
  float amax_t = 0.f;
  if (p.per_tensor) amax_t = __uint_as_float(*p.amax_bits);
  for (long long r = (long long)blockIdx.x * QUANT_REG_WARPS + (threadIdx.x >> 5); r < p.rows;
       r += (long long)gridDim.x * QUANT_REG_WARPS) {
    const uint4* x = p.X + r * nvec;
    uint4 q[NV];
#pragma unroll
    for (int u = 0; u < NV; ++u) {
      const int v = u * 32 + lane;
      q[u] = (v < nvec) ? x[v] : make_uint4(0u, 0u, 0u, 0u);
    }
    float amax = amax_t;
    if (!p.per_tensor) {
      amax = 0.f;
#pragma unroll
      for (int u = 0; u < NV; ++u) amax = fmaxf(amax, q_amax8(q[u]));
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, off));
      if (lane == 0) p.scale[r] = amax > 0.f ? __fdiv_rn(amax, E4M3_MAX) : 1.f;
    }
    const float inv = amax > 0.f ? __fdiv_rn(E4M3_MAX, amax) : 1.f;
    uint2* o = p.Q + r * nvec;
#pragma unroll
    for (int u = 0; u < NV; ++u) {
      const int v = u * 32 + lane;
      if (v < nvec) o[v] = q_pack8(q[u], inv);
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Block-scaled (MX) e4m3: one power-of-two scale per 32 consecutive elements of a row -- the operand format of
// tcgen05.mma.kind::mxf8f6f4.block_scale (next widening of SURVEY section 8(f)-4; reading #26):
//   e    = the smallest integer with amax_blk <= 448 * 2^e, clamped to [-127, 127]   (amax = 0: -127)
//   code = e4m3 nearest (ties to even) to x * 2^-e        scale byte (UE8M0) = e + 127
// Everything is exact: bf16 values are fp32 values, e comes from the exponent and a compare of the significand with 1.75
// (448 = 1.75 * 2^8), the scaling is by powers of two (in two steps, so that 2^127 / 2^-127 never appear as one factor),
// and |x * 2^-e| <= 448.  So codes and exponents must equal the oracle's bit for bit.
// The scale bytes are written in the layout tcgen05.cp (32x128b.warpx4) moves to TMEM unchanged.  Rows are grouped in
// blocks of `blk_rows` (128 for H: the token rows of one CTA; 224 for W: one vocabulary tile), K in blocks of 128
// elements (4 scales).  Region (kb, blk) holds 512-byte pieces of 128 rows each:
//   byte = ((kb * num_blk + blk) * pieces + r / 128) * 512 + (r % 32) * 16 + ((r / 32) % 4) * 4 + (k % 128) / 32,  r = row % blk_rows
struct QuantMxParams {
  const uint4* X;        // bf16 [rows, d] as 16-byte vectors (8 elements)
  uint2* Q;              // e4m3 [rows, d] as 8-byte vectors
  uint8_t* SF;           // scale bytes, layout above (zeroed by the caller: unwritten slots scale zero codes)
  long long rows;
  int d;
  int blk_rows;          // 128 or 224
  int pieces;            // 512-byte pieces per region: ceil(blk_rows / 128)
  int64_t num_blk;       // ceil(rows / blk_rows)
};

__device__ __forceinline__ int mx_exponent(float amax) {   // amax >= 0, finite
  if (amax == 0.f) return -127;
  const uint32_t bits = __float_as_uint(amax);
  const int E = (int)(bits >> 23) - 127;                     // subnormals read as -127: e clamps to -127 either way
  const bool above = (bits & 0x7fffffu) > 0x600000u;         // significand > 1.75
  return max(-127, min(127, E - 8 + (above ? 1 : 0)));
}

__global__ void __launch_bounds__(256) sq_quant_mx_kernel(const QuantMxParams p) {
  const int lane = threadIdx.x & 31;
  const long long warps = (long long)gridDim.x * 8;
  const int nvec = p.d >> 3;                                 // 16-byte vectors per row (d % 16 == 0)
  for (long long row = (long long)blockIdx.x * 8 + (threadIdx.x >> 5); row < p.rows; row += warps) {
    const long long blk = row / p.blk_rows;
    const int r = (int)(row - blk * p.blk_rows);
    const size_t in_region = (size_t)(r >> 7) * 512 + (size_t)(r & 31) * 16 + (size_t)((r >> 5) & 3) * 4;
    constexpr int U = 4;                                     // passes whose loads are issued together (HBM-bound: bytes in flight)
    for (int v0 = 0; v0 < nvec; v0 += 32 * U) {              // a pass: 256 elements = 8 scale blocks; 4 lanes per block
      uint4 xs[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int v = v0 + 32 * u + lane;
        xs[u] = make_uint4(0u, 0u, 0u, 0u);
        if (v < nvec) xs[u] = __ldg(p.X + row * nvec + v);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int v = v0 + 32 * u + lane;
        const uint4 x = xs[u];
        float m = q_amax8(x);
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 1));
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
        const int e = mx_exponent(m);
        const int ea = (-e) / 2, eb = (-e) - ea;             // x * 2^ea * 2^eb, both factors normal floats
        const float fa = __uint_as_float((uint32_t)(ea + 127) << 23), fb = __uint_as_float((uint32_t)(eb + 127) << 23);
        float f[8];
        q_unpack8(x, f);
        uint32_t c[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) c[i] = (uint32_t)__nv_cvt_float_to_fp8(__fmul_rn(__fmul_rn(f[i], fa), fb), __NV_SATFINITE, __NV_E4M3);
        if (v < nvec) {
          uint2 o;
          o.x = c[0] | (c[1] << 8) | (c[2] << 16) | (c[3] << 24);
          o.y = c[4] | (c[5] << 8) | (c[6] << 16) | (c[7] << 24);
          p.Q[row * nvec + v] = o;
          if ((lane & 3) == 0) {
            const int k = v * 8;                             // first element of the scale block
            const size_t region = ((size_t)(k >> 7) * (size_t)p.num_blk + (size_t)blk) * (size_t)p.pieces;
            p.SF[region * 512 + in_region + ((k & 127) >> 5)] = (uint8_t)(e + 127);
          }
        }
      }
    }
  }
}

}  // namespace sq
