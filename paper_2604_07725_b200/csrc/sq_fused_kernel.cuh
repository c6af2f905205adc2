// sq_fused_kernel.cuh -- kernel 1: fused vocabulary GEMM + online softmax statistics (sm_100a).
//
// Steps a1..a5 of the hot path: logits tile Z = H_tile * W_tile^T by
// tcgen05.mma into TMEM (never written to memory), then per row an online logsumexp (m, s), the
// shifted entropy accumulator u = sum e^{z-m}(z-m), the target logit, and a streaming top-k list
// -- the quantities Eq. 3 needs: log p(v_j) = z_(j) - lse.
//
// Persistent, warp-specialised:  warp 0 = TMA producer, warp 1 = MMA issuer, warp 2 = TMEM
// allocator, warps 4..7 = statistics epilogue (thread = TMEM lane = token row).
// Work unit = (token tile of 128*CG rows, vocab chunk = a run of 256-column tiles (224 in the MX variant), FusedParams::chunk_vt);
// a unit's running state lives in registers and is written as a partial state at its end.
#pragma once
#include "sq_ptx.cuh"

namespace sq {

constexpr int BLOCK_M = 128;   // token rows per CTA = TMEM lanes
constexpr int BLOCK_N = 256;   // vocabulary columns per tile = UMMA N
constexpr int BLOCK_K = 64;    // bf16 per k-block: 128 B = one swizzle-128B row (e4m3: 128 elements, BLOCK_K_F8)
constexpr int UMMA_K = 16;     // K per MMA instruction: 32 bytes of each operand row (e4m3: 32 elements)
constexpr int BLOCK_K_F8 = 128;
constexpr int NUM_THREADS = 256;
constexpr int EPI_WARP0 = 4;
constexpr int TMEM_COLS = 512;  // two 256-column accumulator stages
constexpr float NEG_BIG = -1.0e30f;
constexpr float LOG2E_F = 1.4426950408889634f;   // consume32 takes log2(e) times the row's dequantisation scale (1 for bf16)

constexpr int BLOCK_N_MX = 224;   // block-scaled variant: 2 x 224 accumulator columns + 12 columns of scale factors fit TMEM's 512
constexpr int MODE_BF16 = 0, MODE_F8 = 1, MODE_MX = 2;

// AROWS: token rows a stage holds (128; 64 / 32 for decode-shaped runs of at most 64 / 32 rows, single CTA only: the MMA still reads 128
// rows -- the second half is the first rows of the W tile behind it, finite values whose accumulator rows nobody looks at --
// and the 8 / 12 KB saved per stage buy a fifth / sixth stage: an HBM-bound run lives on the W bytes it has in flight).
template <int CG, int MODE = MODE_BF16, int AROWS = 128> struct FusedCfg {
  static constexpr int BN = (MODE == MODE_MX) ? BLOCK_N_MX : BLOCK_N;   // vocabulary columns per tile
  static constexpr int A_BYTES = AROWS * BLOCK_K * 2;                   // 16 KB (8 KB)
  static constexpr int B_ROWS = BN / CG;                                // W rows this CTA stages
  static constexpr int B_BYTES = B_ROWS * BLOCK_K * 2;                  // 32 KB (CG=1) / 16 KB (CG=2); MX: 28 / 14 KB
  // MX: the scale factors of the stage's 128-element k-block: 512 B for this CTA's 128 token rows, 1024 B for ALL the
  // tile's vocabulary rows (every CTA of a pair multiplies its token rows with the whole tile)
  static constexpr int SFA_BYTES = (MODE == MODE_MX) ? 512 : 0;
  static constexpr int SFB_BYTES = (MODE == MODE_MX) ? 1024 : 0;
  static constexpr int STAGE_BYTES = (A_BYTES + B_BYTES + SFA_BYTES + SFB_BYTES + 1023) / 1024 * 1024;
  static constexpr int STAGE_TX = A_BYTES + B_BYTES + SFA_BYTES + SFB_BYTES;   // bytes the TMA loads of a stage deliver
#ifndef SQ_STAGES_PAIR
#define SQ_STAGES_PAIR 6
#endif
  static constexpr int STAGES = (CG == 1) ? (AROWS == 32 ? 6 : (AROWS == 64 ? 5 : 4)) : SQ_STAGES_PAIR;
  static constexpr int BAR_BYTES = 256;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + 1024;  // +1024: manual alignment
  static constexpr int UMMA_M = BLOCK_M * CG;
  static constexpr int TMEM_SFA = 2 * BN;        // MX: TMEM columns of the scale factors, behind the two accumulators
  static constexpr int TMEM_SFB = 2 * BN + 4;
};

constexpr int MAX_CHUNKS = 160;   // vocab chunks per row at most (= FIN_MAX_CHUNKS of the finalize kernel)

struct FusedParams {
  int T, V, d;
  int num_k_blocks;
  int num_vtiles;
  int num_chunks;           // num_gangs * chunks_per_gang
  int m_tiles;
  int num_gangs;
  int gang_size;            // gangs [0, gangs_big) have gang_size + 1 members, the others gang_size
  int gangs_big;
  int chunks_per_gang;      // a gang's vocabulary stripe is cut into this many chunks
  unsigned int* gang_ctr;   // [num_gangs], zeroed before the launch
  unsigned int* region_ctr; // one more counter, zeroed with them: clusters that have finished a region of token tiles
  int region_tiles;         // 0, or: no cluster starts token tile region_tiles * r before every cluster has finished the tiles
  int region_arrivals;      //   below it (r = 1, 2, ...); CTAs that arrive per region (a multiple of every gang size in tiles)
  long long wait_limit;     // clock cycles a wait may last before the kernel traps (0 = wait for ever)
  const int32_t* targets;   // [T]
  float* part_m;            // [C][T]
  float* part_s;            // [C][T]
  float* part_u;            // [C][T]
  float* part_cs;           // [C][T] Kahan residues: the true sums are s - cs and u - cu
  float* part_cu;           // [C][T]
  float* part_topv;         // [C][CAP][T]
  int32_t* part_topi;       // [C][CAP][T]
  float* zt;                // [T] target logit (written by the chunk that owns the target column)
  float* thr_pub;           // null, or [C][T]: chunk c's current thr_j-th best logit of row t (shared top-k bound, below)
  int thr_j, thr_ns;        //   every chunk publishes its thr_j-th best; the bound is the thr_ns-th SMALLEST published value
  const unsigned int* h_ready;   // null, or flags set as H arrives from the host (sq_score_run_host): flag f != 0
  int flag_rows;                 //   <=> rows [0, (f+1) * flag_rows) of H are in device memory
  const float* h_scale;     // FP8 variant: H = Hq * h_scale[row], W = Wq * (*w_scale) with Hq, Wq e4m3 (per-row / per-tensor
  const float* w_scale;     //   scales, DEVICE); null in the bf16 path
  int sf_h_blocks;          // MX variant: 128-row blocks of H in the scale layout (rows of tmap_sfa per k-block)
  int vocab_offset;         // W is rows [vocab_offset, vocab_offset + V) of a larger LM head (vocab-parallel shard):
                            // targets and the reported vocabulary ids are global, columns local
  uint16_t chunk_vt[MAX_CHUNKS + 1];   // chunk c sweeps vocab tiles [chunk_vt[c], chunk_vt[c+1]) (widths differ between gangs)
};

struct Unit { int m_tile; int chunk; };

// Gang scheduling.  The persistent clusters are split into `num_gangs` gangs whose sizes differ by at most one (every
// cluster the device holds belongs to a gang).  Gang i owns vocab chunks [i*r, (i+1)*r), r = chunks_per_gang, and walks
// the token tiles in batches of its own size: member j takes token tile b*size + j of batch b and sweeps the gang's
// chunks for it.  All members sweep the same W chunk at the same time, so each W tile is fetched from HBM once per
// batch and served to the other members from L2; the gangs advance through the token tiles at the same pace (their
// stripe widths are sized for it), so they share the H strips of the current region.
struct GangCtx {
  int ctr;       // index of this gang = index of its barrier counter
  int member;    // position in the gang
  int size;      // clusters in the gang
  int num_iters; // ceil(m_tiles / size) batches x chunks_per_gang chunks
};
__device__ __forceinline__ GangCtx make_gang_ctx(const FusedParams& p, int cluster) {
  GangCtx g;
  const int big_clusters = p.gangs_big * (p.gang_size + 1);
  if (cluster < big_clusters) {
    g.size = p.gang_size + 1;
    g.ctr = cluster / g.size;
    g.member = cluster - g.ctr * g.size;
  } else {
    g.size = p.gang_size;
    const int c = cluster - big_clusters;
    g.ctr = p.gangs_big + c / g.size;
    g.member = c - (c / g.size) * g.size;
  }
  g.num_iters = ((p.m_tiles + g.size - 1) / g.size) * p.chunks_per_gang;
  return g;
}
// iteration `it` of the gang -> this member's unit; false: ragged last batch, the member idles for this iteration
__device__ __forceinline__ bool decode_gang_unit(const FusedParams& p, const GangCtx& gc, int it, Unit& out) {
  const int b = it / p.chunks_per_gang;
  out.chunk = gc.ctr * p.chunks_per_gang + (it - b * p.chunks_per_gang);
  out.m_tile = b * gc.size + gc.member;
  return out.m_tile < p.m_tiles;
}

// Producer-side gang barrier: keeps the members' W streams within L2 reach of one another.  The
// counter only grows (zeroed by the host before the launch); epoch e completes at e * arrivals.
__device__ __forceinline__ void gang_barrier(unsigned int* ctr, unsigned int target, long long limit) {
  __threadfence();
  atomicAdd(ctr, 1u);
  const long long t0 = clock64();
  unsigned int v;
  do {
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
    if (v >= target) break;
    __nanosleep(64);
    if (limit > 0 && clock64() - t0 > limit) __trap();
  } while (true);
}

// H streams in from the host while the kernel runs (sq_score_run_host): rows arrive in ascending order and a copy
// engine sets flag f once rows [0, (f+1) * flag_rows) have landed.  The producer polls before its first load of a unit.
__device__ __forceinline__ void wait_rows_ready(const unsigned int* flag, long long limit) {
  const long long t0 = clock64();
  unsigned int v;
  do {
    asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory");
    if (v != 0u) break;
    __nanosleep(200);
    // the same limit as every other wait of the kernel: the consumers of this producer (full_bar, tfull_bar, the
    // other clusters' gang and region barriers) give up after `limit` anyway, so a longer allowance here could never
    // take effect -- in sq_score_run_host the whole copy of H must land within cfg.wait_seconds
    if (limit > 0 && clock64() - t0 > limit) __trap();
  } while (true);
  asm volatile("fence.proxy.async;" ::: "memory");   // the rows are read through the async proxy (TMA)
}

// Shared top-k bound.  A row's vocabulary is swept by C chunks on C different gangs at about the same time, each
// with its own top-k list, so a chunk that has seen n logits inserts ~k*ln(n/k) times although most of those entries
// cannot survive the merge.  After every tile a chunk publishes its j-th best logit so far, and reads the others':
// if r chunks each hold j logits >= x, and r*j >= k, then x is a lower bound on the row's final k-th best, and a logit
// <= x can be dropped by every chunk (the k logits that prove the bound stay in their owners' lists, so the merged
// top-k VALUES are exact; which of several logits exactly EQUAL to the k-th best is kept may differ).  The bound
// used is the r-th largest = ns-th smallest of the C published values, ns = C - r + 1 <= 3.  Stale or missing values
// only make the bound weaker.  Measured: ~5x fewer list insertions, ~40 % fewer epilogue instructions.
template <int CAP>
__device__ __forceinline__ float shared_topk_bound(const float (&tv)[CAP], const FusedParams& p, int chunk, int row) {
  // thr_j is one of CAP, CAP/2, CAP/4 (host's choice): compile-time slots, so the list stays in registers
  const float mine = (p.thr_j == CAP) ? tv[CAP - 1] : ((p.thr_j == CAP / 2) ? tv[CAP / 2 - 1] : tv[CAP / 4 - 1]);
  float* pub = p.thr_pub + row;
  __stcg(pub + (size_t)chunk * p.T, mine);
  float s0 = 3.0e38f, s1 = 3.0e38f, s2 = 3.0e38f;   // the three smallest published values, ascending
  for (int c = 0; c < p.num_chunks; ++c) {
    const float v = (c == chunk) ? mine : __ldcg(pub + (size_t)c * p.T);
    const float a = fminf(s0, v), b = fmaxf(s0, v);
    const float c1 = fminf(s1, b), d = fmaxf(s1, b);
    s0 = a; s1 = c1; s2 = fminf(s2, d);
  }
  return p.thr_ns == 1 ? s0 : (p.thr_ns == 2 ? s1 : s2);
}

// value of r[i] for a run-time i without local memory: a 5-level select tree.
__device__ __forceinline__ float pick32(const float (&r)[32], int i) {
  float a[16], b[8], c[4], d2[2];
#pragma unroll
  for (int j = 0; j < 16; ++j) a[j] = (i & 1) ? r[2 * j + 1] : r[2 * j];
#pragma unroll
  for (int j = 0; j < 8; ++j) b[j] = (i & 2) ? a[2 * j + 1] : a[2 * j];
#pragma unroll
  for (int j = 0; j < 4; ++j) c[j] = (i & 4) ? b[2 * j + 1] : b[2 * j];
#pragma unroll
  for (int j = 0; j < 2; ++j) d2[j] = (i & 8) ? c[2 * j + 1] : c[2 * j];
  return (i & 16) ? d2[1] : d2[0];
}

// Sorted (descending) insertion of (z, idx) into a register-resident list; the last entry drops out.
template <int CAP>
__device__ __forceinline__ void topk_insert(float (&tv)[CAP], int (&ti)[CAP], float z, int idx) {
#pragma unroll
  for (int j = CAP - 1; j >= 1; --j) {
    const bool above = z > tv[j - 1];   // z belongs above slot j-1: slot j takes slot j-1
    const bool here = z > tv[j];
    ti[j] = above ? ti[j - 1] : (here ? idx : ti[j]);
    tv[j] = above ? tv[j - 1] : (here ? z : tv[j]);
  }
  if (z > tv[0]) { tv[0] = z; ti[0] = idx; }
}

// Per-row running state of one work unit.
template <int CAP> struct RowState {
  float m, s, u, zt;
  float cs, cu;   // Kahan compensation of s and u: a peaked row adds ~1e-7 terms to s ~ 1
  float gthr;     // lower bound on the row's final k-th best logit learnt from the other vocab chunks (-3e38 = none)
  float tv[CAP];
  int ti[CAP];
  __device__ __forceinline__ void reset() {
    m = NEG_BIG; s = 0.f; u = 0.f; zt = 0.f; cs = 0.f; cu = 0.f; gthr = -3.0e38f;
#pragma unroll
    for (int j = 0; j < CAP; ++j) { tv[j] = NEG_BIG; ti[j] = -1; }
  }
};

// Consumes 32 consecutive logits of one row (columns col0 .. col0+31).
template <int CAP>
__device__ __forceinline__ void consume32(RowState<CAP>& st, float (&r)[32], int col0, int V, int tgt, const float LOG2E) {
  if (col0 + 32 > V) {   // ragged vocabulary tail: columns >= V hold TMA zero fill
#pragma unroll
    for (int i = 0; i < 32; ++i) r[i] = (col0 + i < V) ? r[i] : NEG_BIG;
  }
  float g0 = fmaxf(r[0], r[1]), g1 = fmaxf(r[2], r[3]);
#pragma unroll
  for (int i = 4; i < 32; i += 4) {
    g0 = fmaxf(g0, fmaxf(r[i], r[i + 1]));
    g1 = fmaxf(g1, fmaxf(r[i + 2], r[i + 3]));
  }
  const float gmax = fmaxf(g0, g1);
  if (gmax > st.m) {   // new running maximum: rescale s and the shifted entropy sum
    const float dm = st.m - gmax;
    const float sc = ex2_approx(dm * LOG2E);
    st.u = (st.u + dm * st.s) * sc;
    st.cu = (st.cu + dm * st.cs) * sc;
    st.s *= sc;
    st.cs *= sc;
    st.m = gmax;
  }
  const float m = st.m;
  float s0 = 0.f, s1 = 0.f, u0 = 0.f, u1 = 0.f;
#pragma unroll
  for (int i = 0; i < 32; i += 2) {
    const float t0 = r[i] - m, t1 = r[i + 1] - m;
    const float e0 = ex2_approx(t0 * LOG2E), e1 = ex2_approx(t1 * LOG2E);
    s0 += e0; s1 += e1;
    u0 = fmaf(e0, t0, u0); u1 = fmaf(e1, t1, u1);
  }
  {   // compensated accumulation of the group sums
    const float ys = (s0 + s1) - st.cs;
    const float ts = st.s + ys;
    st.cs = (ts - st.s) - ys;
    st.s = ts;
    const float yu = (u0 + u1) - st.cu;
    const float tu = st.u + yu;
    st.cu = (tu - st.u) - yu;
    st.u = tu;
  }

  if ((unsigned)(tgt - col0) < 32u) st.zt = pick32(r, tgt - col0);   // a3: target logit

  // a5: some element of this row beats the current k-th best of this chunk AND the bound from the other chunks
  if (gmax > fmaxf(st.tv[CAP - 1], st.gthr)) {
    uint32_t mask = 0;
    const float thr = fmaxf(st.tv[CAP - 1], st.gthr);
#pragma unroll
    for (int i = 0; i < 32; ++i) mask |= (r[i] > thr) ? (1u << i) : 0u;
    while (mask) {
      const int i = __ffs(mask) - 1;
      mask &= mask - 1;
      const float z = pick32(r, i);
      if (z > st.tv[CAP - 1]) topk_insert<CAP>(st.tv, st.ti, z, col0 + i);   // (the bound itself never rises inside a group)
    }
  }
}

// F8: operands are e4m3 bytes (tcgen05 kind::f8f6f4, 128 elements per 128-byte k-block row); the accumulator is
// Hq.Wq^T and the epilogue works in those units with log2(e) * h_scale[row] * w_scale folded into the exponent's
// multiplier, so the dequantisation costs no instruction per logit; m, u, the list values and the target logit are
// scaled once per row when the partial state is written.
// MX (MODE_MX): e4m3 bytes with one UE8M0 scale per 32 elements of K (tcgen05 kind::mxf8f6f4.block_scale).  The scales of a
// stage arrive by TMA next to the operands (tmap_sfa / tmap_sfb: rows of 512 bytes in the layout tcgen05.cp wants, written
// by sq_quant_mx_kernel), are copied to TMEM by the MMA thread before the stage's four instructions, and the tensor core
// applies them: the accumulator holds the logits themselves, so the epilogue is the bf16 one.  Tiles are 224 columns wide.
// CL = 4: "quad" scheduling (CTA pairs, not for the MX variant).  Four consecutive CTAs -- a quad -- take one 512-row token
// tile, 128 rows each, and sweep the same vocabulary chunk.  The launch asks for clusters of 4 with clusters of 2 as the
// fallback (cudaLaunchAttributePreferredClusterDimension): this part places 33 clusters of 4, and the 16 SMs they cannot
// cover (one TPC per GPC) run the other 4 quads as two independent pairs each.  Which quad got which shape is only known
// at run time (%cluster_nctarank); the work of a CTA does not depend on it, only how W reaches it does:
//   cluster of 4: both pairs are on the SAME W tile at the same time, and every W box is fetched from L2 once for the two
//     pairs -- CTA r loads 64 of the 128 W rows that the CTAs r and r ^ 2 need and multicasts them to both.  L2 -> SM
//     operand traffic per k-block and SM falls from 16 KB (H) + 16 KB (W) to 16 + 8 KB.  A stage is free again when
//     BOTH pairs' MMAs have retired (the commit goes to all four CTAs, the empty barriers count two arrivals).
//   cluster of 2: the pair loads its own 2 x 64 W rows, as in the plain pair kernel.
template <int CG, int CAP, int MODE = MODE_BF16, int CL = CG, int AROWS = 128>
__global__ void __launch_bounds__(NUM_THREADS, 1)
sq_fused_score_kernel(const __grid_constant__ CUtensorMap tmap_h, const __grid_constant__ CUtensorMap tmap_w,
                      const __grid_constant__ CUtensorMap tmap_sfa, const __grid_constant__ CUtensorMap tmap_sfb,
                      const FusedParams p) {
  using Cfg = FusedCfg<CG, MODE, AROWS>;
  static_assert(AROWS == 128 || ((AROWS == 64 || AROWS == 32) && CG == 1), "short token tiles are for single-CTA (decode-shaped) runs");
  constexpr bool F8 = (MODE == MODE_F8);
  constexpr bool MX = (MODE == MODE_MX);
  constexpr int BN = Cfg::BN;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // swizzle-128B: 1024-B aligned tiles
  const uint32_t bar_base = smem_base + Cfg::STAGES * Cfg::STAGE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (Cfg::STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * Cfg::STAGES + 4);
  auto smem_a = [&](int s) { return smem_base + s * Cfg::STAGE_BYTES; };
  auto smem_b = [&](int s) { return smem_base + s * Cfg::STAGE_BYTES + Cfg::A_BYTES; };
  auto smem_sfa = [&](int s) { return smem_base + s * Cfg::STAGE_BYTES + Cfg::A_BYTES + Cfg::B_BYTES; };
  auto smem_sfb = [&](int s) { return smem_base + s * Cfg::STAGE_BYTES + Cfg::A_BYTES + Cfg::B_BYTES + Cfg::SFA_BYTES; };

  const int warp = threadIdx.x >> 5;
  const uint32_t lane = lane_id();
  static_assert(CL == CG || (CL == 4 && CG == 2 && MODE != MODE_MX), "quads are two CTA pairs");
  const uint32_t cl_rank = (CL > 1) ? cluster_ctarank() : 0u;   // rank in the cluster
  const bool mcast = (CL == 4) && cluster_nctarank() == 4;      // this quad is ONE cluster: W boxes are multicast
  const uint32_t unit_rank = (CL == 4) ? (blockIdx.x & 3u) : cl_rank;   // position in the quad / pair: rows 128 * unit_rank of the token tile
  const uint32_t cta_rank = cl_rank & (CG - 1);                 // rank in the CTA pair
  const uint32_t pair_leader = cl_rank & ~1u;                   // cluster rank of this pair's even CTA
  const bool leader = (cta_rank == 0);
  const int cluster = (CL == 4) ? (int)(blockIdx.x >> 2) : ((CL > 1) ? (int)cluster_id_x() : (int)blockIdx.x);
  const GangCtx gc = make_gang_ctx(p, cluster);

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tmap_h);
    prefetch_tensormap(&tmap_w);
    if constexpr (MX) { prefetch_tensormap(&tmap_sfa); prefetch_tensormap(&tmap_sfb); }
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < Cfg::STAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), mcast ? 2 : 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull_bar(a), 1);
      mbar_init(tempty_bar(a), 4 * CG);   // one elected lane per epilogue warp, both CTAs of a pair
    }
    fence_mbar_init();
  }
  if (warp == 2) {
    tmem_alloc<CG>(tmem_slot, TMEM_COLS);
    tmem_relinquish<CG>();
  }
  __syncwarp();
  tc_fence_before();
  if constexpr (CL > 1) cluster_sync_all(); else __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  const int rows_per_unit = BLOCK_M * CL;
  constexpr int BK = (F8 || MX) ? BLOCK_K_F8 : BLOCK_K;   // elements per k-block (128 bytes of every operand row)

  if (warp == 0) {
    // ===================================================================== TMA producer
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      uint32_t stage_tx = Cfg::STAGE_TX * CG;   // the pair leader's barrier counts both CTAs' bytes
      unsigned int epoch = 0;
      for (int gu = 0; gu < gc.num_iters; ++gu) {
        Unit un;
        const bool active = decode_gang_unit(p, gc, gu, un);
        if (p.region_tiles > 0 && gu > 0 && gu % p.chunks_per_gang == 0) {
          // Gangs of different size or stripe width walk the token tiles at slightly different paces.  Over thousands of
          // tiles they drift apart, the H strips they were sharing stop being shared, and the live set outgrows the L2
          // (qwen3_32b: 1.31 TB of DRAM reads per launch, 70 % L2 hits, the clock down to 1.05 GHz under the power cap).
          // A barrier across ALL clusters every region_tiles token tiles bounds the drift to one region's mismatch.
          const int t0 = (gu / p.chunks_per_gang) * gc.size;   // first token tile of this batch
          if (t0 % p.region_tiles == 0)
            gang_barrier(p.region_ctr, (unsigned)(t0 / p.region_tiles) * (unsigned)p.region_arrivals, p.wait_limit);
        }
        if (gc.size > 1) gang_barrier(p.gang_ctr + gc.ctr, (++epoch) * (unsigned)(gc.size * CL), p.wait_limit);
        if (!active) continue;
        const int row0 = un.m_tile * rows_per_unit + (int)unit_rank * BLOCK_M;
        if (p.h_ready != nullptr && row0 < p.T)
          wait_rows_ready(p.h_ready + (min(row0 + BLOCK_M, p.T) - 1) / p.flag_rows, p.wait_limit);
        const int vt0 = p.chunk_vt[un.chunk], vt1 = p.chunk_vt[un.chunk + 1];
        for (int vt = vt0; vt < vt1; ++vt) {
          const int wrow0 = vt * BN + (int)cta_rank * Cfg::B_ROWS;
          for (int kb = 0; kb < p.num_k_blocks; ++kb) {
            mbar_wait(empty_bar(stage), phase ^ 1u, p.wait_limit);
            // MX: scale rows of 512 bytes: [k-block][128-row block of H] and [k-block][vocab tile][2]
            const int sfa_row = kb * p.sf_h_blocks + row0 / BLOCK_M, sfb_row = (kb * p.num_vtiles + vt) * 2;
            if constexpr (CG == 1) {
              mbar_arrive_expect_tx(full_bar(stage), stage_tx);
              tma_load_2d(smem_a(stage), &tmap_h, full_bar(stage), kb * BK, row0);
              tma_load_2d(smem_b(stage), &tmap_w, full_bar(stage), kb * BK, wrow0);
              if constexpr (MX) {
                tma_load_2d(smem_sfa(stage), &tmap_sfa, full_bar(stage), 0, sfa_row);
                tma_load_2d(smem_sfb(stage), &tmap_sfb, full_bar(stage), 0, sfb_row);
              }
            } else {
              const uint32_t bar = mapa(full_bar(stage), pair_leader);
              if (leader) mbar_arrive_expect_tx(full_bar(stage), stage_tx);
              tma_load_2d_pair(smem_a(stage), &tmap_h, bar, kb * BK, row0);
              if constexpr (CL == 4) {   // (tmap_w's boxes are 64 rows high)
                constexpr int HB = Cfg::B_ROWS / 2;
                if (mcast) {             // half of this CTA's W rows, to this CTA and to its counterpart in the other pair
                  const int half = (int)(cl_rank >> 1) * HB;
                  tma_load_2d_pair_mcast(smem_b(stage) + (uint32_t)half * 128u, &tmap_w, full_bar(stage),
                                         (uint16_t)(0x5u << cta_rank), kb * BK, wrow0 + half);
                } else {
                  tma_load_2d_pair(smem_b(stage), &tmap_w, bar, kb * BK, wrow0);
                  tma_load_2d_pair(smem_b(stage) + (uint32_t)HB * 128u, &tmap_w, bar, kb * BK, wrow0 + HB);
                }
              } else {
                tma_load_2d_pair(smem_b(stage), &tmap_w, bar, kb * BK, wrow0);
              }
              if constexpr (MX) {
                tma_load_2d_pair(smem_sfa(stage), &tmap_sfa, bar, 0, sfa_row);
                tma_load_2d_pair(smem_sfb(stage), &tmap_sfb, bar, 0, sfb_row);
              }
            }
            if (++stage == Cfg::STAGES) { stage = 0; phase ^= 1u; }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer (pair leader only)
    if (leader && lane == 0) {
      constexpr uint32_t idesc = MX ? make_idesc_mx(Cfg::UMMA_M, BN)
                                    : (F8 ? make_idesc_e4m3(Cfg::UMMA_M, BN) : make_idesc_bf16(Cfg::UMMA_M, BN));
      int stage = 0; uint32_t phase = 0;
      uint32_t tile = 0;
      for (int gu = 0; gu < gc.num_iters; ++gu) {
        Unit un;
        if (!decode_gang_unit(p, gc, gu, un)) continue;
        const int vt0 = p.chunk_vt[un.chunk], vt1 = p.chunk_vt[un.chunk + 1];
        for (int vt = vt0; vt < vt1; ++vt, ++tile) {
          const uint32_t acc = tile & 1u;
          mbar_wait(tempty_bar(acc), ((tile >> 1) & 1u) ^ 1u, p.wait_limit);   // epilogue drained this accumulator
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + acc * BN;
          for (int kb = 0; kb < p.num_k_blocks; ++kb) {
            mbar_wait(full_bar(stage), phase, p.wait_limit);
            tc_fence_after();
            const uint64_t adesc = make_smem_desc_sw128(smem_a(stage));
            const uint64_t bdesc = make_smem_desc_sw128(smem_b(stage));
            if constexpr (MX) {
              // this k-block's scales: 4 columns for the 128 token rows, 8 for the tile's vocabulary rows.  The copies run in
              // the tensor pipe, in order with the MMAs: 3 x ~16 clk against 4 x 112 clk of MMA per k-block (measured: 48.0 ms
              // with them, 43.5 ms without; alternating between two or four sets of columns changes nothing, so one set)
              tmem_cp_32x128b_warpx4<CG>(tmem_base + Cfg::TMEM_SFA, make_smem_desc_sf(smem_sfa(stage)));
              tmem_cp_32x128b_warpx4<CG>(tmem_base + Cfg::TMEM_SFB, make_smem_desc_sf(smem_sfb(stage)));
              tmem_cp_32x128b_warpx4<CG>(tmem_base + Cfg::TMEM_SFB + 4, make_smem_desc_sf(smem_sfb(stage) + 512));
            }
#pragma unroll
            for (int k = 0; k < BLOCK_K / UMMA_K; ++k) {
              // +32 B per UMMA_K step inside the 128-B swizzle row: +2 in the (addr >> 4) field
              if constexpr (MX) umma_mx<CG>(d_tmem, adesc + 2u * k, bdesc + 2u * k, idesc_mx_sf(idesc, k), tmem_base + Cfg::TMEM_SFA,
                                            tmem_base + Cfg::TMEM_SFB, (kb | k) != 0 ? 1u : 0u);
              else if constexpr (F8) umma_f8<CG>(d_tmem, adesc + 2u * k, bdesc + 2u * k, idesc, (kb | k) != 0 ? 1u : 0u);
              else umma_bf16<CG>(d_tmem, adesc + 2u * k, bdesc + 2u * k, idesc, (kb | k) != 0 ? 1u : 0u);
            }
            umma_commit<CG>(empty_bar(stage), mcast ? (uint16_t)0xF : (uint16_t)0x3);   // smem slot free once these MMAs retire
            if (++stage == Cfg::STAGES) { stage = 0; phase ^= 1u; }
          }
          umma_commit<CG>(tfull_bar(acc), (uint16_t)(0x3u << pair_leader));   // accumulator ready for the epilogue (this pair's)
        }
      }
    }
  } else if (warp >= EPI_WARP0) {
    // ===================================================================== statistics epilogue
    const int q = warp & 3;                       // TMEM lane quarter this warp may read
    const int row_in_tile = q * 32 + (int)lane;
    const uint32_t lane_addr = tmem_base + (static_cast<uint32_t>(q * 32) << 16);
    const uint32_t tempty_remote = (CG == 2) ? mapa(tempty_bar(0), pair_leader) : tempty_bar(0);
    RowState<CAP> st;
    uint32_t tile = 0;
    for (int gu = 0; gu < gc.num_iters; ++gu) {
      Unit un;
      if (!decode_gang_unit(p, gc, gu, un)) continue;
      const int row = un.m_tile * rows_per_unit + (int)unit_rank * BLOCK_M + row_in_tile;
      const int vt0 = p.chunk_vt[un.chunk], vt1 = p.chunk_vt[un.chunk + 1];
      int tgt = (row < p.T) ? __ldg(p.targets + row) : -1;
      tgt = (tgt >= p.vocab_offset) ? tgt - p.vocab_offset : -1;   // local column, or out of range
      st.reset();
      float deq = 1.f;                             // F8: accumulator units -> logits for this row
      if constexpr (F8) deq = ((row < p.T) ? __ldg(p.h_scale + row) : 1.f) * __ldg(p.w_scale);
      const float l2e = F8 ? LOG2E_F * deq : LOG2E_F;
      for (int vt = vt0; vt < vt1; ++vt, ++tile) {
        const uint32_t acc = tile & 1u;
        mbar_wait(tfull_bar(acc), (tile >> 1) & 1u, p.wait_limit);
        tc_fence_after();
        const int colbase = vt * BN;
        int ngroups = min(BN, p.V - colbase + 31) >> 5;   // 32-column groups with a valid column
        if (AROWS < BLOCK_M && q * 32 >= AROWS) ngroups = 0;   // this warp's TMEM lanes hold no token rows
        for (int g = 0; g < ngroups; ++g) {
          float r[32];
          tmem_ld_32x32(lane_addr + acc * BN + g * 32, r);
          tmem_ld_wait();
          consume32<CAP>(st, r, colbase + g * 32, p.V, tgt, l2e);
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          if constexpr (CG == 2) mbar_arrive_cluster(tempty_remote + 8u * acc);
          else mbar_arrive(tempty_bar(acc));
        }
        if (p.thr_pub != nullptr && row < p.T && vt + 1 < vt1)
          st.gthr = fmaxf(st.gthr, shared_topk_bound<CAP>(st.tv, p, un.chunk, row));
      }
      if (row < p.T) {
        const size_t o = (size_t)un.chunk * p.T + row;
        p.part_m[o] = st.m * deq;                  // deq == 1 in the bf16 path: exact
        p.part_s[o] = st.s;
        p.part_u[o] = st.u * deq;
        p.part_cs[o] = st.cs;
        p.part_cu[o] = st.cu * deq;
#pragma unroll
        for (int j = 0; j < CAP; ++j) {
          const size_t oj = ((size_t)un.chunk * CAP + j) * p.T + row;
          p.part_topv[oj] = st.tv[j] * deq;
          p.part_topi[oj] = st.ti[j] < 0 ? -1 : st.ti[j] + p.vocab_offset;
        }
        const int c0 = vt0 * BN;
        if (tgt >= c0 && tgt < min(vt1 * BN, p.V)) p.zt[row] = st.zt * deq;
      }
    }
  }

  // ----------------------------------------------------------------------- teardown
  __syncwarp();
  tc_fence_before();
  if constexpr (CL > 1) cluster_sync_all(); else __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<CG>(tmem_base, TMEM_COLS);
  }
}

}  // namespace sq
