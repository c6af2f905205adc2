// sq_score_api.cu -- C ABI of libsq_score.so (include/sq_score.h): context, planning, TMA tensor
// maps and kernel launches.  No torch types, no CPU fallback.
#include "../../include/sq_score.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "sq_finalize_kernel.cuh"
#include "sq_fused_kernel.cuh"
#include "sq_prepare_kernel.cuh"
#include "sq_quant_kernel.cuh"
#include "sq_reduce_kernel.cuh"
#include "sq_route_kernel.cuh"

#define SQ_VERSION 100

struct sq_score_ctx {
  sq_score_config cfg;
  int num_sms = 0;
  int cap_max = 0;          // top-k capacity the workspace is sized for
  int chunks_max = 0;       // largest num_chunks the workspace holds
  int64_t launches = 0;
  char err[512] = {0};
  // partial states
  float* part_m = nullptr; float* part_s = nullptr; float* part_u = nullptr;
  float* part_cs = nullptr; float* part_cu = nullptr;
  float* part_topv = nullptr; int32_t* part_topi = nullptr; float* zt = nullptr;
  unsigned int* gang_ctr = nullptr;
  float* thr_pub = nullptr;   // [THR_MAX_CHUNKS][max_tokens] shared top-k bounds (sq_fused_kernel.cuh)
  // per-token scratch (used when the caller passes NULL per-token outputs)
  float* tok_lse = nullptr; float* tok_lp = nullptr; float* tok_ent = nullptr; float* tok_conf = nullptr;
  // kernel 2 workspace
  unsigned int* amax_bits = nullptr;   // per-tensor amax of sq_score_quantize_fp8
  int* seq_done = nullptr;   // [max_seqs] per-sequence tile counters of the single-launch reduction (zero between runs)
  int* tile_base = nullptr; int* tile_seq = nullptr; float4* red_sum = nullptr; float* red_min = nullptr; int64_t red_tiles_max = 0;
  // staging for sq_score_run_host
  void* h_stage = nullptr; int32_t* tgt_stage = nullptr; int32_t* cu_stage = nullptr; float* seq_stage = nullptr;
  // sq_score_run_host streams H in on its own copy stream while kernel 1 runs: one flag per block of rows
  cudaStream_t copy_stream = nullptr; cudaEvent_t ev_fork = nullptr, ev_small = nullptr, ev_join = nullptr;
  unsigned int* h_flags = nullptr; unsigned int* one_host = nullptr;
  // driver entry point for tensor-map encoding
  void* encode_fn = nullptr;
  // optional per-kernel timing (sq_score_set_profiling): events around kernel 1, finalize, kernel 2
  int profiling = 0; int ev_valid = 0; int debug_flags = 0;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
};

static thread_local char g_create_err[512] = {0};

static int set_err(sq_score_ctx* ctx, int code, const char* fmt, ...) {
  char* dst = ctx ? ctx->err : g_create_err;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return code;
}

#define SQ_CUDA(ctx, call)                                                                   \
  do {                                                                                       \
    cudaError_t e_ = (call);                                                                 \
    if (e_ != cudaSuccess)                                                                   \
      return set_err(ctx, SQ_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                     __FILE__, __LINE__);                                                    \
  } while (0)

constexpr int THR_MAX_CHUNKS = 16;   // the shared top-k bound is used for 2..16 vocab chunks per row

static int topk_cap_for(int k) { return k <= 8 ? 8 : (k <= 20 ? 20 : 32); }
static inline int64_t cdiv64(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ------------------------------------------------------------------------------------------ plan
// Work decomposition.  A unit sweeps `tiles_per_chunk` vocab tiles for one
// token tile; units are ordered [group of group_m token tiles][chunk][tile in group] and handed to
// the persistent clusters round-robin, so ~num_clusters consecutive units are in flight: group_m
// token strips (H stays in L2) x ~num_clusters/group_m chunks (each W tile is read from HBM once
// per group and shared through L2 by the group_m units that sweep it in lockstep).
static int make_plan(const sq_score_config* cfg, int64_t T, int k, int num_sms, sq_score_plan_t* pl) {
  if (!cfg || !pl || T < 0 || cfg->d <= 0 || cfg->vocab <= 0 || k < 1 || k > SQ_MAX_K) return SQ_ERR_INVALID_ARG;
  if (num_sms <= 0) num_sms = 148;
  // default: CTA pairs (UMMA M = 256); a decode-shaped run of at most 128 rows fits one CTA's 128 TMEM
  // lanes, so single-CTA UMMA (M = 128) halves the wasted MMA rows and lets all 148 SMs stream W
  const int cg = (cfg->cta_group == 1) ? 1 : (cfg->cta_group == 2 ? 2 : ((T > 0 && T <= 128) ? 1 : 2));
  memset(pl, 0, sizeof(*pl));
  pl->cta_group = cg;
  pl->rows_per_tile = 128 * cg;
  pl->m_tiles = (int)cdiv64(T, pl->rows_per_tile);
  pl->num_vtiles = (int)cdiv64(cfg->vocab, 256);
  pl->num_k_blocks = (int)cdiv64(cfg->d, 64);
  pl->num_clusters = std::max(1, num_sms / cg);
  pl->topk_cap = topk_cap_for(k);
  // gang size: group_m clusters sweep one W chunk together, never more than there are token tiles or
  // clusters.  Default 12 (measured on B200 against 8 / 10 / 14 / 16 / 24: +1.5 % at qwen3_8b, +2.7 % at
  // gpt_oss, neutral at qwen3_4b -- W is read from HBM once per 12 token tiles instead of 8 and the
  // planner then needs fewer, longer vocab chunks)
  int G = cfg->group_m > 0 ? cfg->group_m : 12;
  G = std::max(1, std::min(G, std::min(std::max(1, pl->m_tiles), pl->num_clusters)));
  pl->group_m = G;
  pl->num_gangs = pl->num_clusters / G;
  const int GB = pl->num_clusters - pl->num_gangs * G;   // clusters left over: one smaller gang B
  pl->gang_b_size = GB;
  const int M = pl->m_tiles;
  const int max_chunks = std::min((int)sq::FIN_MAX_CHUNKS, pl->num_vtiles);
  // cost of a plan = the slower gang class, in tile-times: rounds x (unit length + fill/drain)
  auto eval = [&](int c, int m_b, double* cost_out) {
    const int tpc = (int)cdiv64(pl->num_vtiles, c);
    const int ce = (int)cdiv64(pl->num_vtiles, tpc);
    const int64_t rounds_a = cdiv64(cdiv64(M - m_b, G) * ce, pl->num_gangs);
    const int64_t rounds_b = m_b > 0 ? cdiv64(m_b, GB) * ce : 0;
    *cost_out = (double)std::max(rounds_a, rounds_b) * (tpc + 0.75);   // 0.75 tile-times of fill/drain per unit
    return ce;
  };
  int best_c = 1, best_mb = 0;
  if (M > 0) {
    // The gangs in flight work on ceil(num_gangs / C) different token groups, i.e. about
    // num_clusters / C token strips of rows_per_tile x d bf16 are re-read from L2 for every vocab
    // tile.  Keep that hot set under ~40 MB of the 126 MB L2 (measured: beyond ~50 MB the strips
    // start to miss and HBM traffic and power go up), then minimise the cost above over the number
    // of chunks and the number of token tiles handed to gang B; ties -> fewer chunks, smaller B.
    const double strip_mb = (double)pl->rows_per_tile * cfg->d * 2.0 / 1e6;
    const int c_l2 = (int)std::ceil(pl->num_gangs * G * strip_mb / 40.0);
    // decode-shaped runs (fewer token groups than gangs) split the vocabulary further so that every
    // cluster streams its own slice of W: up to one chunk per gang
    const int64_t groups = cdiv64(M, G);
    int c_hi = std::min(max_chunks, groups * 16 < pl->num_gangs ? (int)cdiv64(pl->num_gangs, groups) : 16);
    int c_lo = std::max(1, std::min(c_hi, c_l2));
    if (cfg->num_chunks > 0) c_lo = c_hi = std::min(cfg->num_chunks, max_chunks);
    const int mb_hi = GB > 0 ? std::min(M - 1, (int)(3.0 * M * GB / pl->num_clusters) + GB) : 0;
    double best_cost = 1e300;
    for (int c = c_lo; c <= c_hi; ++c) {
      for (int m_b = 0; m_b <= mb_hi; ++m_b) {
        double cost;
        const int ce = eval(c, m_b, &cost);
        if (ce < c_lo && c < c_hi) break;   // rounding merged chunks below the L2 bound
        if (cost < best_cost - 1e-9) { best_cost = cost; best_c = c; best_mb = m_b; }
      }
    }
  } else if (cfg->num_chunks > 0) {
    best_c = std::min(cfg->num_chunks, max_chunks);
  }
  pl->tiles_per_chunk = (int)cdiv64(pl->num_vtiles, best_c);
  pl->num_chunks = (int)cdiv64(pl->num_vtiles, pl->tiles_per_chunk);
  pl->num_units = pl->m_tiles * pl->num_chunks;
  pl->m_split = M - best_mb;
  pl->num_gang_units = (int)cdiv64(pl->m_split, G) * pl->num_chunks;
  pl->num_gang_units_b = best_mb > 0 ? (int)cdiv64(best_mb, GB) * pl->num_chunks : 0;
  return SQ_OK;
}

extern "C" int sq_score_plan(const sq_score_config* cfg, int64_t num_tokens, int k, int num_sms,
                             sq_score_plan_t* plan) {
  return make_plan(cfg, num_tokens, k, num_sms, plan);
}

extern "C" int sq_score_version(void) { return SQ_VERSION; }

extern "C" const char* sq_score_error_string(int code) {
  switch (code) {
    case SQ_OK: return "SQ_OK";
    case SQ_ERR_INVALID_ARG: return "SQ_ERR_INVALID_ARG";
    case SQ_ERR_UNSUPPORTED: return "SQ_ERR_UNSUPPORTED";
    case SQ_ERR_CUDA: return "SQ_ERR_CUDA";
    case SQ_ERR_NOMEM: return "SQ_ERR_NOMEM";
    default: return "SQ_ERR_UNKNOWN";
  }
}

extern "C" const char* sq_score_last_error(const sq_score_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

extern "C" int64_t sq_score_launch_count(const sq_score_ctx* ctx) { return ctx ? ctx->launches : 0; }

// ------------------------------------------------------------------------------------------ create / destroy
static int64_t ws_rows_for(const sq_score_config& cfg) {
  const int64_t small_t = std::min<int64_t>(cfg.max_tokens, 4096);
  int64_t rows = std::max<int64_t>((int64_t)sq::FIN_MAX_CHUNKS * small_t, 16 * cfg.max_tokens);
  if (cfg.num_chunks > 0) rows = std::max<int64_t>(rows, (int64_t)std::min(cfg.num_chunks, (int)sq::FIN_MAX_CHUNKS) * cfg.max_tokens);
  return rows;
}

extern "C" int sq_score_destroy(sq_score_ctx* ctx) {
  if (!ctx) return SQ_OK;
  cudaSetDevice(ctx->cfg.device);
  void* bufs[] = {ctx->amax_bits, ctx->seq_done, ctx->thr_pub, ctx->gang_ctr, ctx->part_cs, ctx->part_cu, ctx->part_m, ctx->part_s, ctx->part_u, ctx->part_topv, ctx->part_topi, ctx->zt,
                  ctx->tok_lse, ctx->tok_lp, ctx->tok_ent, ctx->tok_conf, ctx->tile_base, ctx->tile_seq, ctx->red_sum,
                  ctx->red_min, ctx->h_stage, ctx->tgt_stage, ctx->cu_stage, ctx->seq_stage};
  int rc = SQ_OK;
  for (void* b : bufs)
    if (b && cudaFree(b) != cudaSuccess) rc = SQ_ERR_CUDA;
  for (cudaEvent_t e : ctx->ev)
    if (e) cudaEventDestroy(e);
  for (cudaEvent_t e : {ctx->ev_fork, ctx->ev_small, ctx->ev_join})
    if (e) cudaEventDestroy(e);
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  if (ctx->h_flags && cudaFree(ctx->h_flags) != cudaSuccess) rc = SQ_ERR_CUDA;
  if (ctx->one_host) cudaFreeHost(ctx->one_host);
  delete ctx;
  return rc;
}

template <typename T>
static int ws_alloc(sq_score_ctx* ctx, T** p, int64_t count) {
  if (count <= 0) count = 1;
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), (size_t)count * sizeof(T));
  if (e != cudaSuccess) {
    *p = nullptr;
    cudaGetLastError();
    return set_err(ctx, e == cudaErrorMemoryAllocation ? SQ_ERR_NOMEM : SQ_ERR_CUDA,
                   "workspace allocation of %lld bytes failed: %s", (long long)(count * (int64_t)sizeof(T)),
                   cudaGetErrorString(e));
  }
  return SQ_OK;
}

extern "C" int sq_score_create(const sq_score_config* cfg, sq_score_ctx** out) {
  if (out) *out = nullptr;
  if (!cfg || !out) return set_err(nullptr, SQ_ERR_INVALID_ARG, "null argument");
  if (cfg->d <= 0 || cfg->vocab <= 0 || cfg->max_tokens <= 0 || cfg->max_seqs <= 0)
    return set_err(nullptr, SQ_ERR_INVALID_ARG, "d, vocab, max_tokens and max_seqs must be positive");
  if (cfg->max_k < 1 || cfg->max_k > SQ_MAX_K)
    return set_err(nullptr, SQ_ERR_INVALID_ARG, "max_k must be in 1..%d", SQ_MAX_K);
  if (cfg->cta_group < 0 || cfg->cta_group > 2 || cfg->num_chunks < 0 || cfg->group_m < 0 || (cfg->flags & ~SQ_FLAG_REDUCE_ONLY))
    return set_err(nullptr, SQ_ERR_INVALID_ARG, "cta_group must be 0, 1 or 2; num_chunks, group_m >= 0");
  if (cfg->d % 8 != 0)
    return set_err(nullptr, SQ_ERR_UNSUPPORTED, "d = %d is not a multiple of 8 (TMA needs 16-byte row strides)", cfg->d);
  if (cfg->max_tokens >= (1LL << 31) - 16384)
    return set_err(nullptr, SQ_ERR_UNSUPPORTED, "max_tokens must be below 2^31 - 16384");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return set_err(nullptr, SQ_ERR_CUDA, "no CUDA device available: %s (this library has no CPU fallback)",
                   e == cudaSuccess ? "device count is 0" : cudaGetErrorString(e));
  }
  if (cfg->device < 0 || cfg->device >= ndev) return set_err(nullptr, SQ_ERR_INVALID_ARG, "device %d out of range", cfg->device);
  cudaDeviceProp prop;
  SQ_CUDA(nullptr, cudaGetDeviceProperties(&prop, cfg->device));
  if (prop.major != 10)
    return set_err(nullptr, SQ_ERR_UNSUPPORTED, "device %d is sm_%d%d; the kernels are built for sm_100a only", cfg->device,
                   prop.major, prop.minor);
  SQ_CUDA(nullptr, cudaSetDevice(cfg->device));

  sq_score_ctx* ctx = new (std::nothrow) sq_score_ctx();
  if (!ctx) return set_err(nullptr, SQ_ERR_NOMEM, "host allocation failed");
  ctx->cfg = *cfg;
  ctx->num_sms = prop.multiProcessorCount;
  if (const char* lim = getenv("SQ_SCORE_MAX_SMS"))   // experiments only: plan for fewer SMs
    if (atoi(lim) >= 2 && atoi(lim) < ctx->num_sms) ctx->num_sms = atoi(lim);
  ctx->cap_max = topk_cap_for(cfg->max_k);
  if (const char* dbg = getenv("SQ_SCORE_DEBUG")) ctx->debug_flags = atoi(dbg);

  cudaDriverEntryPointQueryResult qres;
  e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ctx->encode_fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !ctx->encode_fn) {
    set_err(nullptr, SQ_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    delete ctx;
    return SQ_ERR_CUDA;
  }

  const bool reduce_only = (cfg->flags & SQ_FLAG_REDUCE_ONLY) != 0;
  const int64_t rows = reduce_only ? 1 : ws_rows_for(*cfg);
  const int64_t T = cfg->max_tokens;
  ctx->red_tiles_max = cdiv64(T, sq::RED_TILE) + 2 * (int64_t)cfg->max_seqs + 1;
  int rc = SQ_OK;
  auto A = [&](int r) { if (rc == SQ_OK && r != SQ_OK) rc = r; };
  A(ws_alloc(ctx, &ctx->part_m, rows));
  A(ws_alloc(ctx, &ctx->part_s, rows));
  A(ws_alloc(ctx, &ctx->part_u, rows));
  A(ws_alloc(ctx, &ctx->part_cs, rows));
  A(ws_alloc(ctx, &ctx->part_cu, rows));
  A(ws_alloc(ctx, &ctx->part_topv, rows * ctx->cap_max));
  A(ws_alloc(ctx, &ctx->part_topi, rows * ctx->cap_max));
  A(ws_alloc(ctx, &ctx->zt, reduce_only ? 1 : T));
  A(ws_alloc(ctx, &ctx->gang_ctr, 256));
  A(ws_alloc(ctx, &ctx->thr_pub, reduce_only ? 1 : (int64_t)THR_MAX_CHUNKS * T));
  A(ws_alloc(ctx, &ctx->tok_lse, reduce_only ? 1 : T));
  A(ws_alloc(ctx, &ctx->tok_lp, reduce_only ? 1 : T));
  A(ws_alloc(ctx, &ctx->tok_ent, reduce_only ? 1 : T));
  A(ws_alloc(ctx, &ctx->tok_conf, reduce_only ? 1 : T));
  A(ws_alloc(ctx, &ctx->tile_base, (int64_t)cfg->max_seqs + 1));
  A(ws_alloc(ctx, &ctx->amax_bits, 1));
  A(ws_alloc(ctx, &ctx->seq_done, (int64_t)cfg->max_seqs));
  if (rc == SQ_OK && cudaMemset(ctx->seq_done, 0, (size_t)cfg->max_seqs * sizeof(int)) != cudaSuccess) rc = SQ_ERR_CUDA;
  A(ws_alloc(ctx, &ctx->red_sum, ctx->red_tiles_max));
  A(ws_alloc(ctx, &ctx->tile_seq, ctx->red_tiles_max));
  A(ws_alloc(ctx, &ctx->red_min, ctx->red_tiles_max));
  A(ws_alloc(ctx, &ctx->seq_stage, 4 * (int64_t)cfg->max_seqs));
  if (rc != SQ_OK) {
    memcpy(g_create_err, ctx->err, sizeof(g_create_err));
    sq_score_destroy(ctx);
    return rc;
  }
  // opt in to the large dynamic shared memory of every fused-kernel instantiation
#define SQ_SET_SMEM(CG, CAP)                                                                                   \
  if (cudaFuncSetAttribute(sq::sq_fused_score_kernel<CG, CAP>, cudaFuncAttributeMaxDynamicSharedMemorySize,    \
                           sq::FusedCfg<CG>::SMEM_BYTES) != cudaSuccess) rc = SQ_ERR_CUDA;
  SQ_SET_SMEM(1, 8) SQ_SET_SMEM(1, 20) SQ_SET_SMEM(1, 32) SQ_SET_SMEM(2, 8) SQ_SET_SMEM(2, 20) SQ_SET_SMEM(2, 32)
#undef SQ_SET_SMEM
#define SQ_SET_SMEM8(CG, CAP)                                                                                      \
  if (cudaFuncSetAttribute(sq::sq_fused_score_kernel<CG, CAP, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,  \
                           sq::FusedCfg<CG>::SMEM_BYTES) != cudaSuccess) rc = SQ_ERR_CUDA;
  SQ_SET_SMEM8(1, 8) SQ_SET_SMEM8(1, 20) SQ_SET_SMEM8(1, 32) SQ_SET_SMEM8(2, 8) SQ_SET_SMEM8(2, 20) SQ_SET_SMEM8(2, 32)
#undef SQ_SET_SMEM8
  for (const void* f : {(const void*)sq::sq_reduce_fused_kernel<true>, (const void*)sq::sq_reduce_fused_kernel<false>})
    if (cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             sq::RED_SMEM_BYTES + (sq::RED_FUSED_MAX_SEQS + 1) * (int)sizeof(int)) != cudaSuccess) rc = SQ_ERR_CUDA;
  if (rc != SQ_OK) {
    set_err(nullptr, rc, "cudaFuncSetAttribute(MaxDynamicSharedMemorySize) failed: %s", cudaGetErrorString(cudaGetLastError()));
    sq_score_destroy(ctx);
    return rc;
  }
  *out = ctx;
  return SQ_OK;
}

// ------------------------------------------------------------------------------------------ tensor maps
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// bf16 [rows, d] row-major -> boxes of {64 columns (128 B, swizzle-128B), box_rows rows}; out-of-range
// rows and columns are zero filled.
static int make_tmap(sq_score_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int d, int box_rows, bool f8 = false) {
  const cuuint64_t dims[2] = {(cuuint64_t)d, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)d * (f8 ? 1 : 2)};
  const cuuint32_t box[2] = {(cuuint32_t)(f8 ? sq::BLOCK_K_F8 : sq::BLOCK_K), (cuuint32_t)box_rows};   // 128 bytes wide
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = reinterpret_cast<encode_tiled_fn>(ctx->encode_fn)(
      map, f8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_err(ctx, SQ_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  return SQ_OK;
}

// ------------------------------------------------------------------------------------------ launches
template <int CG, int CAP, bool F8 = false>
static cudaError_t launch_fused(const sq_score_plan_t& pl, int num_sms, const CUtensorMap& th, const CUtensorMap& tw,
                                const sq::FusedParams& fp, cudaStream_t st) {
  // every launched cluster belongs to a gang; gang B is launched only if it was given token tiles
  const int clusters = pl.num_gangs * pl.group_m + (pl.num_gang_units_b > 0 ? pl.gang_b_size : 0);
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)(clusters * CG));
  lc.blockDim = dim3(sq::NUM_THREADS);
  lc.dynamicSmemBytes = sq::FusedCfg<CG>::SMEM_BYTES;
  lc.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = CG; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  lc.attrs = at;
  lc.numAttrs = 1;
  (void)num_sms;
  return cudaLaunchKernelEx(&lc, sq::sq_fused_score_kernel<CG, CAP, F8>, th, tw, fp);
}

// Launch with programmatic stream serialization: the kernel is scheduled while its predecessor drains and waits in
// cudaGridDependencySynchronize() for its results.
template <typename K, typename P>
static cudaError_t launch_pdl(K kernel, dim3 grid, dim3 block, size_t smem, cudaStream_t st, const P& params) {
  cudaLaunchConfig_t lc = {};
  lc.gridDim = grid; lc.blockDim = block; lc.dynamicSmemBytes = smem; lc.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = 1;
  return cudaLaunchKernelEx(&lc, kernel, params);
}

static int launch_reduce(sq_score_ctx* ctx, sq::ReduceParams& rp, cudaStream_t st) {
  if (rp.B <= 0) return SQ_OK;
  // 16-byte loads need 16-byte aligned arrays (tiles start on multiples of 4 tokens)
  rp.vec = ((((uintptr_t)rp.lp | (uintptr_t)rp.ent | (uintptr_t)rp.conf | (uintptr_t)rp.targets) & 15) == 0) ? 1 : 0;
  const int64_t tiles = cdiv64(rp.T, sq::RED_TILE) + 2 * (int64_t)rp.B;   // upper bound on sum_b ceil((L_b + 3) / RED_TILE)
  // Single launch (sq_reduce_kernel.cuh) when the whole problem is one wave of CTAs -- the scoring pipeline's case, a few
  // dozen tiles, where the three launches are pure latency (20 -> 8 us).  On large inputs the three-launch form is 2x
  // faster (measured 0.099 vs 0.218 ms on 3.6e7 tokens: a persistent CTA pays the fence + atomic + barriers per tile in
  // series), so it stays.  SQ_SCORE_DEBUG bit 5 / bit 6 force the three-launch / single-launch form (tests).
  const size_t fused_smem = sq::RED_SMEM_BYTES + (size_t)(rp.B + 1) * sizeof(int);
  const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(6, (size_t)(220 * 1024) / (fused_smem + 1024)));
  const bool one_wave = tiles <= (int64_t)ctx->num_sms * per_sm && rp.B <= 2048;
  if (rp.B <= sq::RED_FUSED_MAX_SEQS && !(ctx->debug_flags & 32) && (one_wave || (ctx->debug_flags & 64))) {
    rp.seq_done = ctx->seq_done;
    const size_t smem = fused_smem;
    const dim3 grid((unsigned)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)ctx->num_sms * per_sm)));
    if (rp.targets) SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_fused_kernel<true>, grid, dim3(sq::RED_THREADS), smem, st, rp));
    else SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_fused_kernel<false>, grid, dim3(sq::RED_THREADS), smem, st, rp));
    ctx->launches += 1;
    SQ_CUDA(ctx, cudaGetLastError());
    return SQ_OK;
  }
  SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_tile_scan_kernel, dim3(1), dim3(1024), 0, st, rp));
  ctx->launches += 1;
  if (rp.T > 0) {
    // programmatic dependent launch: tile_part's CTAs are scheduled while tile_scan drains and wait
    // in cudaGridDependencySynchronize() for its results
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)tiles);
    lc.blockDim = dim3(sq::RED_THREADS);
    lc.dynamicSmemBytes = sq::RED_SMEM_BYTES;
    lc.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = at;
    lc.numAttrs = 1;
    if (rp.targets) SQ_CUDA(ctx, cudaLaunchKernelEx(&lc, sq::sq_reduce_tile_part_kernel<true>, rp));
    else SQ_CUDA(ctx, cudaLaunchKernelEx(&lc, sq::sq_reduce_tile_part_kernel<false>, rp));
    lc.gridDim = dim3((unsigned)cdiv64(rp.B, 4));
    lc.blockDim = dim3(128);
    lc.dynamicSmemBytes = 0;
    SQ_CUDA(ctx, cudaLaunchKernelEx(&lc, sq::sq_reduce_seq_final_kernel, rp));
    ctx->launches += 2;
  }
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
}

extern "C" int sq_score_reduce(sq_score_ctx* ctx, const float* target_logprob, const float* entropy, const float* conf,
                               const int32_t* targets, const int32_t* cu_seqlens, int64_t num_tokens, int num_seqs,
                               int window, float* seq_mean_logprob, float* seq_mean_entropy, float* seq_mean_conf,
                               float* seq_min_window_conf, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_tokens < 0 || num_seqs < 0 || window < 1) return set_err(ctx, SQ_ERR_INVALID_ARG, "T, B >= 0 and window >= 1 required");
  if (num_tokens > ctx->cfg.max_tokens || num_seqs > ctx->cfg.max_seqs)
    return set_err(ctx, SQ_ERR_INVALID_ARG, "T = %lld / B = %d exceed max_tokens / max_seqs of this ctx", (long long)num_tokens, num_seqs);
  if (num_seqs == 0) return SQ_OK;
  if (!cu_seqlens || !seq_mean_logprob || !seq_mean_entropy || !seq_mean_conf || !seq_min_window_conf ||
      (num_tokens > 0 && (!target_logprob || !entropy || !conf)))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  sq::ReduceParams rp = {};
  rp.T = num_tokens; rp.B = num_seqs; rp.V = ctx->cfg.vocab; rp.window = window;
  rp.lp = target_logprob; rp.ent = entropy; rp.conf = conf; rp.targets = targets; rp.cu = cu_seqlens;
  rp.tile_base = ctx->tile_base; rp.tile_seq = ctx->tile_seq; rp.part_sum = ctx->red_sum; rp.part_min = ctx->red_min;
  rp.out_lp = seq_mean_logprob; rp.out_ent = seq_mean_entropy; rp.out_conf = seq_mean_conf; rp.out_min = seq_min_window_conf;
  return launch_reduce(ctx, rp, static_cast<cudaStream_t>(stream));
}

// Packed partial state of one vocab-parallel shard, in 4-byte words (the exchange unit of sq_score_run_shard /
// sq_score_merge_shards): m[T] s[T] u[T] cs[T] cu[T] topv[cap][T] topi[cap][T] zt[T] -- one chunk in the layout the
// finalize kernel merges.
static int64_t shard_state_words(int64_t T, int cap) { return (6 + 2 * (int64_t)cap) * T; }
static void set_state_pointers(sq::FinalizeParams& f, float* base, int64_t T, int cap, bool as_output) {
  float* m = base; float* s_ = base + T; float* u = base + 2 * T; float* cs = base + 3 * T; float* cu = base + 4 * T;
  float* tv = base + 5 * T; int32_t* ti = reinterpret_cast<int32_t*>(base + (5 + (int64_t)cap) * T);
  float* zt = base + (5 + 2 * (int64_t)cap) * T;
  if (as_output) {
    f.out_m = m; f.out_s = s_; f.out_u = u; f.out_cs = cs; f.out_cu = cu; f.out_topv = tv; f.out_topi = ti; f.out_zt = zt;
  } else {
    f.part_m = m; f.part_s = s_; f.part_u = u; f.part_cs = cs; f.part_cu = cu; f.part_topv = tv; f.part_topi = ti; f.zt = zt;
  }
}

// h_ready / flag_rows: null / 0, or the arrival flags of an H that is still streaming in (sq_score_run_host)
static int run_impl(sq_score_ctx* ctx, const void* H, const void* W, const int32_t* targets,
                    const int32_t* cu_seqlens, int num_tokens, int num_seqs, int k, int window,
                    const sq_score_outputs* o, void* stream, const unsigned int* h_ready, int flag_rows,
                    int vocab_offset = 0, float* shard_state = nullptr, const float* h_scale = nullptr,
                    const float* w_scale = nullptr) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (!o && !shard_state) return set_err(ctx, SQ_ERR_INVALID_ARG, "outputs is null");
  static const sq_score_outputs no_outputs = {};
  if (!o) o = &no_outputs;
  if (ctx->cfg.flags & SQ_FLAG_REDUCE_ONLY) return set_err(ctx, SQ_ERR_INVALID_ARG, "ctx was created with SQ_FLAG_REDUCE_ONLY");
  const int T = num_tokens, V = ctx->cfg.vocab, d = ctx->cfg.d;
  int B = num_seqs;
  if (T < 0 || B < 0) return set_err(ctx, SQ_ERR_INVALID_ARG, "negative T or B");
  if (T > ctx->cfg.max_tokens || B > ctx->cfg.max_seqs)
    return set_err(ctx, SQ_ERR_INVALID_ARG, "T = %d / B = %d exceed max_tokens / max_seqs of this ctx", T, B);
  if (k < 1 || k > ctx->cfg.max_k || k > V) return set_err(ctx, SQ_ERR_INVALID_ARG, "k = %d outside 1..min(max_k, V)", k);
  if (window < 1) return set_err(ctx, SQ_ERR_INVALID_ARG, "window must be >= 1");
  if (shard_state) B = 0;   // a shard run stops at the merged partial state
  if (B > 0 && (!cu_seqlens || !o->seq_mean_logprob || !o->seq_mean_entropy || !o->seq_mean_conf || !o->seq_min_window_conf))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "cu_seqlens and the four per-sequence outputs are required");
  if (T > 0 && (!H || !W || !targets)) return set_err(ctx, SQ_ERR_INVALID_ARG, "H, W and targets are required");
  if (T > 0 && (((uintptr_t)H & 15) || ((uintptr_t)W & 15))) return set_err(ctx, SQ_ERR_INVALID_ARG, "H and W must be 16-byte aligned");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  float* lse = o->lse ? o->lse : ctx->tok_lse;
  float* lp = o->target_logprob ? o->target_logprob : ctx->tok_lp;
  float* ent = o->entropy ? o->entropy : ctx->tok_ent;
  float* conf = o->conf ? o->conf : ctx->tok_conf;

  if (T > 0) {
    const bool f8 = h_scale != nullptr;
    sq_score_plan_t pl;
    sq_score_config pc = ctx->cfg;
    if (f8) pc.d = (d + 1) / 2;   // an e4m3 k-block is 128 elements: the plan sees half as many k-blocks
    make_plan(&pc, T, k, ctx->num_sms, &pl);
    const int64_t rows = ws_rows_for(ctx->cfg);
    if ((int64_t)pl.num_chunks * T > rows) {   // workspace bound: fewer, longer chunks
      pc.num_chunks = (int)std::max<int64_t>(1, rows / T);
      make_plan(&pc, T, k, ctx->num_sms, &pl);
    }
    if (pl.topk_cap > ctx->cap_max) return set_err(ctx, SQ_ERR_INVALID_ARG, "k exceeds the ctx's max_k capacity");
    CUtensorMap th, tw;
    if (f8 && d % 16 != 0) return set_err(ctx, SQ_ERR_UNSUPPORTED, "the FP8 variant needs d %% 16 == 0 (TMA 16-byte row strides)");
    int rc = make_tmap(ctx, &th, H, T, d, (ctx->debug_flags & 4) ? sq::BLOCK_M / 2 : sq::BLOCK_M, f8);
    if (rc != SQ_OK) return rc;
    rc = make_tmap(ctx, &tw, W, V, d, (sq::BLOCK_N / pl.cta_group) / ((ctx->debug_flags & 2) ? 2 : 1), f8);
    if (rc != SQ_OK) return rc;

    sq::FusedParams fp = {};
    fp.T = T; fp.V = V; fp.d = d;
    fp.num_k_blocks = pl.num_k_blocks; fp.num_vtiles = pl.num_vtiles; fp.tiles_per_chunk = pl.tiles_per_chunk;
    fp.num_chunks = pl.num_chunks; fp.m_tiles = pl.m_tiles; fp.group_m = pl.group_m;
    fp.num_gangs = pl.num_gangs; fp.num_gang_units = pl.num_gang_units; fp.gang_ctr = ctx->gang_ctr;
    fp.m_split = pl.m_split; fp.gang_b_size = pl.gang_b_size; fp.num_gang_units_b = pl.num_gang_units_b;
    // the gang barrier counters only matter when some gang has more than one member (not in decode-shaped plans)
    if (pl.group_m > 1 || (pl.num_gang_units_b > 0 && pl.gang_b_size > 1))
      SQ_CUDA(ctx, cudaMemsetAsync(ctx->gang_ctr, 0, 256 * sizeof(unsigned int), st));
    fp.targets = targets;
    fp.part_m = ctx->part_m; fp.part_s = ctx->part_s; fp.part_u = ctx->part_u;
    fp.part_cs = ctx->part_cs; fp.part_cu = ctx->part_cu;
    fp.part_topv = ctx->part_topv; fp.part_topi = ctx->part_topi; fp.zt = ctx->zt;
    fp.debug_flags = ctx->debug_flags;
    fp.vocab_offset = vocab_offset;
    fp.h_scale = h_scale; fp.w_scale = w_scale;
    fp.h_ready = h_ready; fp.flag_rows = flag_rows;
    if (pl.num_chunks >= 2 && pl.num_chunks <= THR_MAX_CHUNKS && !(ctx->debug_flags & 16)) {
      // every chunk publishes its j-th best, j one of cap/4, cap/2, cap (compile-time list slots); r = ceil(k / j)
      // chunks holding j logits above x prove the bound, and the kernel takes the ns-th smallest published value,
      // ns = C - r + 1 capped at 3 (a larger r only weakens the bound)
      const int C = pl.num_chunks, cap = pl.topk_cap;
      int j = cap;
      for (int cand : {cap / 4, cap / 2})
        if (cand >= 1 && (k + cand - 1) / cand <= C) { j = cand; break; }
      const int r = (k + j - 1) / j;
      fp.thr_pub = ctx->thr_pub; fp.thr_j = j; fp.thr_ns = std::min(3, C - r + 1);
      // "nothing published": a finite value below every logit (bytes 0xFE -> -1.7e38)
      SQ_CUDA(ctx, cudaMemsetAsync(ctx->thr_pub, 0xFE, (size_t)C * T * sizeof(float), st));
    }
    cudaError_t e;
    if (ctx->profiling) cudaEventRecord(ctx->ev[0], st);
    const int sel = pl.cta_group * 100 + pl.topk_cap + (f8 ? 1000 : 0);
    switch (sel) {
      case 1108: e = launch_fused<1, 8, true>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 1120: e = launch_fused<1, 20, true>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 1132: e = launch_fused<1, 32, true>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 1208: e = launch_fused<2, 8, true>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 1220: e = launch_fused<2, 20, true>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 1232: e = launch_fused<2, 32, true>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 108: e = launch_fused<1, 8>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 120: e = launch_fused<1, 20>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 132: e = launch_fused<1, 32>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 208: e = launch_fused<2, 8>(pl, ctx->num_sms, th, tw, fp, st); break;
      case 220: e = launch_fused<2, 20>(pl, ctx->num_sms, th, tw, fp, st); break;
      default: e = launch_fused<2, 32>(pl, ctx->num_sms, th, tw, fp, st); break;
    }
    if (e != cudaSuccess) return set_err(ctx, SQ_ERR_CUDA, "fused kernel launch failed: %s", cudaGetErrorString(e));
    if (ctx->profiling) cudaEventRecord(ctx->ev[1], st);

    sq::FinalizeParams fin = {};
    fin.T = T; fin.V = V; fin.k = k; fin.cap = pl.topk_cap; fin.num_chunks = pl.num_chunks;
    fin.targets = targets;
    fin.part_m = ctx->part_m; fin.part_s = ctx->part_s; fin.part_u = ctx->part_u;
    fin.part_cs = ctx->part_cs; fin.part_cu = ctx->part_cu;
    fin.part_topv = ctx->part_topv; fin.part_topi = ctx->part_topi; fin.zt = ctx->zt;
    fin.lse = lse; fin.target_logprob = lp; fin.entropy = ent; fin.conf = conf;
    fin.topk_logprob = o->topk_logprob; fin.topk_index = o->topk_index;
    fin.chunks_per_rank = pl.num_chunks; fin.rank_stride = 0; fin.num_ranks = 1;
    const dim3 fgrid((unsigned)cdiv64(T, sq::FIN_WARPS)), fblock(sq::FIN_WARPS * 32);
    const dim3 fgrid8((unsigned)cdiv64(T, sq::FIN_WARPS * 4));   // 8 lanes per row: four rows per warp
    const bool lpr8 = pl.num_chunks <= 8 && !(ctx->debug_flags & 128);
    if (shard_state && lpr8) {
      set_state_pointers(fin, shard_state, T, pl.topk_cap, /*as_output=*/true);
      SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<1, true, 8>, fgrid8, fblock, 0, st, fin));
    } else if (!shard_state && lpr8) {
      SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<1, false, 8>, fgrid8, fblock, 0, st, fin));
    } else if (shard_state) {   // vocab-parallel shard: the merged state goes out in the packed exchange layout
      set_state_pointers(fin, shard_state, T, pl.topk_cap, /*as_output=*/true);
      if (pl.num_chunks <= 32) SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<1, true>, fgrid, fblock, 0, st, fin));
      else SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<sq::FIN_MAX_NL, true>, fgrid, fblock, 0, st, fin));
    } else if (pl.num_chunks <= 32) {
      SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<1, false>, fgrid, fblock, 0, st, fin));
    } else {
      SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<sq::FIN_MAX_NL, false>, fgrid, fblock, 0, st, fin));
    }
    ctx->launches += 2;
    SQ_CUDA(ctx, cudaGetLastError());
    if (ctx->profiling) cudaEventRecord(ctx->ev[2], st);
  }
  if (B > 0) {
    sq::ReduceParams rp = {};
    rp.T = T; rp.B = B; rp.V = V; rp.window = window;
    rp.lp = lp; rp.ent = ent; rp.conf = conf; rp.targets = targets; rp.cu = cu_seqlens;
    rp.tile_base = ctx->tile_base; rp.tile_seq = ctx->tile_seq; rp.part_sum = ctx->red_sum; rp.part_min = ctx->red_min;
    rp.out_lp = o->seq_mean_logprob; rp.out_ent = o->seq_mean_entropy; rp.out_conf = o->seq_mean_conf;
    rp.out_min = o->seq_min_window_conf;
    const int rc = launch_reduce(ctx, rp, st);
    if (rc != SQ_OK) return rc;
    if (ctx->profiling && T > 0) { cudaEventRecord(ctx->ev[3], st); ctx->ev_valid = 1; }
  }
  return SQ_OK;
}

extern "C" int sq_score_run(sq_score_ctx* ctx, const void* H, const void* W, const int32_t* targets,
                            const int32_t* cu_seqlens, int num_tokens, int num_seqs, int k, int window,
                            const sq_score_outputs* o, void* stream) {
  return run_impl(ctx, H, W, targets, cu_seqlens, num_tokens, num_seqs, k, window, o, stream, nullptr, 0);
}

// ------------------------------------------------------------------------------------------ FP8 variant (8(f)-4)
extern "C" int sq_score_quantize_fp8(sq_score_ctx* ctx, const void* X, int64_t num_rows, int per_tensor, void* q_out,
                                     float* scale_out, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_rows < 0) return set_err(ctx, SQ_ERR_INVALID_ARG, "negative row count");
  if (num_rows == 0) return SQ_OK;
  if (!X || !q_out || !scale_out) return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)X & 15) || ((uintptr_t)q_out & 7)) return set_err(ctx, SQ_ERR_INVALID_ARG, "X must be 16-byte and q_out 8-byte aligned");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  sq::QuantParams qp = {};
  qp.X = static_cast<const uint4*>(X); qp.Q = static_cast<uint2*>(q_out); qp.scale = scale_out;
  qp.amax_bits = ctx->amax_bits; qp.rows = num_rows; qp.d = ctx->cfg.d; qp.per_tensor = per_tensor ? 1 : 0;
  const unsigned ctas = (unsigned)std::min<int64_t>(cdiv64(num_rows, sq::QUANT_WARPS), (int64_t)ctx->num_sms * 8);
  if (per_tensor) {
    SQ_CUDA(ctx, cudaMemsetAsync(ctx->amax_bits, 0, sizeof(unsigned int), st));
    sq::sq_quant_amax_kernel<<<(unsigned)ctx->num_sms * 8, 256, 0, st>>>(qp);
    sq::sq_quant_scale_kernel<<<1, 1, 0, st>>>(qp);
    ctx->launches += 2;
  }
  const unsigned ctas_reg = (unsigned)std::min<int64_t>(cdiv64(num_rows, sq::QUANT_REG_WARPS), (int64_t)ctx->num_sms * 8);
  const int nv = (int)cdiv64(qp.d, 256);
  if (nv <= 4) sq::sq_quant_rows_reg_kernel<4><<<ctas_reg, sq::QUANT_REG_WARPS * 32, 0, st>>>(qp);
  else if (nv <= 8) sq::sq_quant_rows_reg_kernel<8><<<ctas_reg, sq::QUANT_REG_WARPS * 32, 0, st>>>(qp);
  else if (nv <= 12) sq::sq_quant_rows_reg_kernel<12><<<ctas_reg, sq::QUANT_REG_WARPS * 32, 0, st>>>(qp);
  else if (nv <= 16) sq::sq_quant_rows_reg_kernel<16><<<ctas_reg, sq::QUANT_REG_WARPS * 32, 0, st>>>(qp);
  else if (nv <= 24) sq::sq_quant_rows_reg_kernel<24><<<ctas_reg, sq::QUANT_REG_WARPS * 32, 0, st>>>(qp);
  else sq::sq_quant_rows_kernel<<<ctas, sq::QUANT_WARPS * 32, 0, st>>>(qp);   // d > 6144
  ctx->launches += 1;
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
}

extern "C" int sq_score_run_fp8(sq_score_ctx* ctx, const void* Hq, const float* h_scale, const void* Wq, const float* w_scale,
                                const int32_t* targets, const int32_t* cu_seqlens, int num_tokens, int num_seqs, int k,
                                int window, const sq_score_outputs* outputs, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_tokens > 0 && (!h_scale || !w_scale)) return set_err(ctx, SQ_ERR_INVALID_ARG, "h_scale and w_scale are required");
  return run_impl(ctx, Hq, Wq, targets, cu_seqlens, num_tokens, num_seqs, k, window, outputs, stream, nullptr, 0, 0, nullptr,
                  h_scale, w_scale);
}

// ------------------------------------------------------------------------------------------ vocab-parallel (8(f)-4)
extern "C" int64_t sq_score_shard_state_bytes(int64_t num_tokens, int k) {
  if (num_tokens < 0 || k < 1 || k > SQ_MAX_K) return -1;
  return shard_state_words(num_tokens, topk_cap_for(k)) * 4;
}

extern "C" int sq_score_run_shard(sq_score_ctx* ctx, const void* H, const void* W_shard, int vocab_offset,
                                  const int32_t* targets, int num_tokens, int k, void* state_out, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (vocab_offset < 0) return set_err(ctx, SQ_ERR_INVALID_ARG, "vocab_offset must be >= 0");
  if (num_tokens > 0 && !state_out) return set_err(ctx, SQ_ERR_INVALID_ARG, "state_out is null");
  if (num_tokens == 0) return SQ_OK;
  return run_impl(ctx, H, W_shard, targets, nullptr, num_tokens, 0, k, 1, nullptr, stream, nullptr, 0, vocab_offset,
                  static_cast<float*>(state_out));
}

extern "C" int sq_score_merge_shards(sq_score_ctx* ctx, const void* states, int num_shards, const int32_t* vocab_starts,
                                     const int32_t* targets, const int32_t* cu_seqlens, int num_tokens, int num_seqs,
                                     int k, int window, const sq_score_outputs* o, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (!o) return set_err(ctx, SQ_ERR_INVALID_ARG, "outputs is null");
  if (ctx->cfg.flags & SQ_FLAG_REDUCE_ONLY) return set_err(ctx, SQ_ERR_INVALID_ARG, "ctx was created with SQ_FLAG_REDUCE_ONLY");
  const int T = num_tokens, B = num_seqs;
  if (T < 0 || B < 0 || T > ctx->cfg.max_tokens || B > ctx->cfg.max_seqs)
    return set_err(ctx, SQ_ERR_INVALID_ARG, "T / B out of range for this ctx");
  if (num_shards < 1 || num_shards > 32 || !vocab_starts) return set_err(ctx, SQ_ERR_INVALID_ARG, "1..32 shards with their vocabulary starts required");
  for (int r = 0; r < num_shards; ++r)
    if (vocab_starts[r] < 0 || vocab_starts[r + 1] < vocab_starts[r]) return set_err(ctx, SQ_ERR_INVALID_ARG, "vocab_starts must be non-decreasing from >= 0");
  const int Vg = vocab_starts[num_shards];
  if (k < 1 || k > ctx->cfg.max_k || k > Vg) return set_err(ctx, SQ_ERR_INVALID_ARG, "k = %d outside 1..min(max_k, V)", k);
  if (window < 1) return set_err(ctx, SQ_ERR_INVALID_ARG, "window must be >= 1");
  if (B > 0 && (!cu_seqlens || !o->seq_mean_logprob || !o->seq_mean_entropy || !o->seq_mean_conf || !o->seq_min_window_conf))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "cu_seqlens and the four per-sequence outputs are required");
  if (T > 0 && (!states || !targets)) return set_err(ctx, SQ_ERR_INVALID_ARG, "states and targets are required");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  float* lse = o->lse ? o->lse : ctx->tok_lse;
  float* lp = o->target_logprob ? o->target_logprob : ctx->tok_lp;
  float* ent = o->entropy ? o->entropy : ctx->tok_ent;
  float* conf = o->conf ? o->conf : ctx->tok_conf;
  if (T > 0) {
    const int cap = topk_cap_for(k);
    sq::FinalizeParams fin = {};
    fin.T = T; fin.V = Vg; fin.k = k; fin.cap = cap; fin.num_chunks = num_shards;
    fin.chunks_per_rank = 1; fin.rank_stride = shard_state_words(T, cap); fin.num_ranks = num_shards;
    for (int r = 0; r <= num_shards; ++r) fin.vstart[r] = vocab_starts[r];
    fin.targets = targets;
    set_state_pointers(fin, const_cast<float*>(static_cast<const float*>(states)), T, cap, /*as_output=*/false);
    fin.lse = lse; fin.target_logprob = lp; fin.entropy = ent; fin.conf = conf;
    fin.topk_logprob = o->topk_logprob; fin.topk_index = o->topk_index;
    if (num_shards <= 8)
      SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<1, false, 8>, dim3((unsigned)cdiv64(T, sq::FIN_WARPS * 4)), dim3(sq::FIN_WARPS * 32), 0, st, fin));
    else
      SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<1, false>, dim3((unsigned)cdiv64(T, sq::FIN_WARPS)), dim3(sq::FIN_WARPS * 32), 0, st, fin));
    ctx->launches += 1;
    SQ_CUDA(ctx, cudaGetLastError());
  }
  if (B > 0) {
    sq::ReduceParams rp = {};
    rp.T = T; rp.B = B; rp.V = Vg; rp.window = window;
    rp.lp = lp; rp.ent = ent; rp.conf = conf; rp.targets = targets; rp.cu = cu_seqlens;
    rp.tile_base = ctx->tile_base; rp.tile_seq = ctx->tile_seq; rp.part_sum = ctx->red_sum; rp.part_min = ctx->red_min;
    rp.out_lp = o->seq_mean_logprob; rp.out_ent = o->seq_mean_entropy; rp.out_conf = o->seq_mean_conf;
    rp.out_min = o->seq_min_window_conf;
    const int rc = launch_reduce(ctx, rp, st);
    if (rc != SQ_OK) return rc;
  }
  return SQ_OK;
}

extern "C" int sq_score_set_profiling(sq_score_ctx* ctx, int enable) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  if (enable)
    for (auto& e : ctx->ev)
      if (!e) SQ_CUDA(ctx, cudaEventCreate(&e));
  ctx->profiling = enable ? 1 : 0;
  ctx->ev_valid = 0;
  return SQ_OK;
}

extern "C" int sq_score_kernel_times(sq_score_ctx* ctx, float* ms3) {
  if (!ctx || !ms3) return SQ_ERR_INVALID_ARG;
  if (!ctx->profiling || !ctx->ev_valid) return set_err(ctx, SQ_ERR_INVALID_ARG, "no profiled run recorded");
  SQ_CUDA(ctx, cudaEventSynchronize(ctx->ev[3]));
  for (int i = 0; i < 3; ++i) SQ_CUDA(ctx, cudaEventElapsedTime(&ms3[i], ctx->ev[i], ctx->ev[i + 1]));
  return SQ_OK;
}

// H staging [max_tokens, d] bf16, allocated on first use: the landing buffer of sq_score_run_host and the output of the
// prepare step inside sq_score_run_x
static int ensure_h_stage(sq_score_ctx* ctx) {
  if (ctx->h_stage) return SQ_OK;
  return ws_alloc(ctx, reinterpret_cast<uint8_t**>(&ctx->h_stage), ctx->cfg.max_tokens * (int64_t)ctx->cfg.d * 2);
}

// ------------------------------------------------------------------------------------------ prepare (8(f)-2)
extern "C" int sq_score_prepare(sq_score_ctx* ctx, const void* X, int num_rows, const int32_t* pos, int num_tokens,
                                const void* gain, float eps, void* H_out, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_rows < 0 || num_tokens < 0 || !(eps >= 0.f)) return set_err(ctx, SQ_ERR_INVALID_ARG, "negative size or eps");
  if (num_tokens == 0) return SQ_OK;
  if (!X || !gain || !H_out || num_rows == 0) return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument or no source rows");
  if (!pos && num_tokens > num_rows) return set_err(ctx, SQ_ERR_INVALID_ARG, "pos is null (identity) but T > num_rows");
  if (((uintptr_t)X & 15) || ((uintptr_t)gain & 15) || ((uintptr_t)H_out & 15))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "X, gain and H_out must be 16-byte aligned");
  if (pos && H_out == X) return set_err(ctx, SQ_ERR_INVALID_ARG, "in-place operation needs pos == NULL");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  sq::PrepareParams pp = {};
  pp.X = static_cast<const uint4*>(X); pp.pos = pos; pp.gain = static_cast<const uint4*>(gain);
  pp.H = static_cast<uint4*>(H_out); pp.T = num_tokens; pp.N = num_rows; pp.d = ctx->cfg.d; pp.eps = eps;
  const int64_t ctas = std::min<int64_t>(cdiv64(num_tokens, sq::PREP_WARPS), (int64_t)ctx->num_sms * 8);
  const int64_t ctas_reg = std::min<int64_t>(cdiv64(num_tokens, sq::PREP_REG_WARPS), (int64_t)ctx->num_sms * 6);
  const dim3 grid((unsigned)ctas_reg), block(sq::PREP_REG_WARPS * 32);
  cudaStream_t pst = static_cast<cudaStream_t>(stream);
  const int nv = (int)cdiv64(pp.d, 256);   // 16-byte vectors per lane when the row lives in registers
  const size_t gain_smem = (size_t)pp.d * 2;   // <= 12 KB
  if (nv <= 4 && !(ctx->debug_flags & 8)) sq::sq_prepare_reg_kernel<4><<<grid, block, gain_smem, pst>>>(pp);
  else if (nv <= 8 && !(ctx->debug_flags & 8)) sq::sq_prepare_reg_kernel<8><<<grid, block, gain_smem, pst>>>(pp);
  else if (nv <= 12 && !(ctx->debug_flags & 8)) sq::sq_prepare_reg_kernel<12><<<grid, block, gain_smem, pst>>>(pp);
  else if (nv <= 16 && !(ctx->debug_flags & 8)) sq::sq_prepare_reg_kernel<16><<<grid, block, gain_smem, pst>>>(pp);
  else if (nv <= 24 && !(ctx->debug_flags & 8)) sq::sq_prepare_reg_kernel<24><<<grid, block, gain_smem, pst>>>(pp);
  else sq::sq_prepare_kernel<<<(unsigned)ctas, sq::PREP_WARPS * 32, 0, pst>>>(pp);   // d > 6144: two passes
  ctx->launches += 1;
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
}

extern "C" int sq_score_run_x(sq_score_ctx* ctx, const void* X, int num_rows, const int32_t* pos, const void* gain, float eps,
                              const void* W, const int32_t* targets, const int32_t* cu_seqlens, int num_tokens, int num_seqs,
                              int k, int window, const sq_score_outputs* outputs, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (ctx->cfg.flags & SQ_FLAG_REDUCE_ONLY) return set_err(ctx, SQ_ERR_INVALID_ARG, "ctx was created with SQ_FLAG_REDUCE_ONLY");
  if (num_tokens < 0 || num_tokens > ctx->cfg.max_tokens) return set_err(ctx, SQ_ERR_INVALID_ARG, "T out of range for this ctx");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = ensure_h_stage(ctx);
  if (rc != SQ_OK) return rc;
  rc = sq_score_prepare(ctx, X, num_rows, pos, num_tokens, gain, eps, ctx->h_stage, stream);
  if (rc != SQ_OK) return rc;
  return run_impl(ctx, ctx->h_stage, W, targets, cu_seqlens, num_tokens, num_seqs, k, window, outputs, stream, nullptr, 0);
}

constexpr int HOST_FLAG_ROWS_MIN = 2048;   // rows of H per arrival flag (doubled until a run needs at most ...
constexpr int HOST_FLAGS_PER_RUN = 256;    // ... this many flags)

extern "C" int sq_score_run_host(sq_score_ctx* ctx, const void* H_host, const void* W_dev, const int32_t* targets_host,
                                 const int32_t* cu_seqlens_host, int num_tokens, int num_seqs, int k, int window,
                                 float* seq_out_host, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  const int T = num_tokens, B = num_seqs;
  if (T < 0 || B < 0 || T > ctx->cfg.max_tokens || B > ctx->cfg.max_seqs)
    return set_err(ctx, SQ_ERR_INVALID_ARG, "T / B out of range for this ctx");
  if ((T > 0 && (!H_host || !W_dev || !targets_host)) || (B > 0 && (!cu_seqlens_host || !seq_out_host)))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument");
  if (ctx->cfg.flags & SQ_FLAG_REDUCE_ONLY) return set_err(ctx, SQ_ERR_INVALID_ARG, "ctx was created with SQ_FLAG_REDUCE_ONLY");
  if (k < 1 || k > ctx->cfg.max_k || k > ctx->cfg.vocab || window < 1)   // before any copy is enqueued
    return set_err(ctx, SQ_ERR_INVALID_ARG, "k = %d outside 1..min(max_k, V) or window = %d < 1", k, window);
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (!ctx->copy_stream) {   // staging is allocated on first use: only callers of the host form pay for it
    int rc = ensure_h_stage(ctx);
    if (rc == SQ_OK) rc = ws_alloc(ctx, &ctx->tgt_stage, ctx->cfg.max_tokens);
    if (rc == SQ_OK) rc = ws_alloc(ctx, &ctx->cu_stage, (int64_t)ctx->cfg.max_seqs + 1);
    if (rc == SQ_OK) rc = ws_alloc(ctx, &ctx->h_flags, HOST_FLAGS_PER_RUN);
    if (rc != SQ_OK) return rc;
    SQ_CUDA(ctx, cudaHostAlloc(reinterpret_cast<void**>(&ctx->one_host), sizeof(unsigned int), cudaHostAllocDefault));
    *ctx->one_host = 1u;
    SQ_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    SQ_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
    SQ_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_small, cudaEventDisableTiming));
    SQ_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming));
  }
  // H streams in on the ctx's copy stream in blocks of `flag_rows` rows, ascending, each followed by a 4-byte
  // copy that raises the block's flag; kernel 1 starts as soon as targets and cu_seqlens are in and its producers
  // wait for the flag of the rows they are about to load, so the transfer hides behind the GEMM.
  int flag_rows = HOST_FLAG_ROWS_MIN;
  while (cdiv64(T, flag_rows) > HOST_FLAGS_PER_RUN) flag_rows *= 2;
  const int nflags = (int)cdiv64(T, flag_rows);
  cudaStream_t cs = ctx->copy_stream;
  if (T > 0) SQ_CUDA(ctx, cudaMemsetAsync(ctx->h_flags, 0, (size_t)nflags * sizeof(unsigned int), st));
  SQ_CUDA(ctx, cudaEventRecord(ctx->ev_fork, st));         // staging buffers are free once earlier work on `st` is done
  SQ_CUDA(ctx, cudaStreamWaitEvent(cs, ctx->ev_fork, 0));
  if (T > 0) SQ_CUDA(ctx, cudaMemcpyAsync(ctx->tgt_stage, targets_host, (size_t)T * 4, cudaMemcpyHostToDevice, cs));
  if (B > 0) SQ_CUDA(ctx, cudaMemcpyAsync(ctx->cu_stage, cu_seqlens_host, (size_t)(B + 1) * 4, cudaMemcpyHostToDevice, cs));
  SQ_CUDA(ctx, cudaEventRecord(ctx->ev_small, cs));
  const size_t row_bytes = (size_t)ctx->cfg.d * 2;
  for (int f = 0; f < nflags; ++f) {
    const int64_t r0 = (int64_t)f * flag_rows, r1 = std::min<int64_t>(T, r0 + flag_rows);
    SQ_CUDA(ctx, cudaMemcpyAsync(static_cast<uint8_t*>(ctx->h_stage) + r0 * row_bytes,
                                 static_cast<const uint8_t*>(H_host) + r0 * row_bytes, (size_t)(r1 - r0) * row_bytes,
                                 cudaMemcpyHostToDevice, cs));
    SQ_CUDA(ctx, cudaMemcpyAsync(ctx->h_flags + f, ctx->one_host, sizeof(unsigned int), cudaMemcpyHostToDevice, cs));
  }
  SQ_CUDA(ctx, cudaEventRecord(ctx->ev_join, cs));
  SQ_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_small, 0));
  sq_score_outputs o = {};
  o.seq_mean_logprob = ctx->seq_stage;
  o.seq_mean_entropy = ctx->seq_stage + B;
  o.seq_mean_conf = ctx->seq_stage + 2 * (size_t)B;
  o.seq_min_window_conf = ctx->seq_stage + 3 * (size_t)B;
  int rc = run_impl(ctx, ctx->h_stage, W_dev, ctx->tgt_stage, ctx->cu_stage, T, B, k, window, &o, stream,
                    T > 0 ? ctx->h_flags : nullptr, flag_rows);
  SQ_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_join, 0));   // also on the error path: `st` never runs ahead of the copies
  if (rc != SQ_OK) return rc;
  if (B > 0) SQ_CUDA(ctx, cudaMemcpyAsync(seq_out_host, ctx->seq_stage, (size_t)4 * B * sizeof(float), cudaMemcpyDeviceToHost, st));
  return SQ_OK;
}

// ------------------------------------------------------------------------------------------ routing (8(f)-1)
extern "C" int sq_score_route(sq_score_ctx* ctx, const float* seq_conf, int num_seqs, const int32_t* group_members,
                              const int32_t* group_offsets, int num_problems, int num_groups, int group_size,
                              int max_groups_per_problem, const uint8_t* lite_mask, float percentile,
                              float* group_fitness, float* theta, int32_t* route, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_problems < 0 || num_groups < 0 || num_seqs < 0 || group_size < 1 || max_groups_per_problem < 0)
    return set_err(ctx, SQ_ERR_INVALID_ARG, "negative size or group_size < 1");
  if (!(percentile >= 0.f && percentile <= 100.f)) return set_err(ctx, SQ_ERR_INVALID_ARG, "percentile must be in [0, 100]");
  if (max_groups_per_problem > sq::ROUTE_MAX_GROUPS)
    return set_err(ctx, SQ_ERR_UNSUPPORTED, "at most %d groups per problem", sq::ROUTE_MAX_GROUPS);
  if (num_problems == 0) return SQ_OK;
  if (!group_offsets || !theta || (num_groups > 0 && (!seq_conf || !group_members || !group_fitness || !route)))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  sq::RouteParams rp = {};
  rp.seq_conf = seq_conf; rp.group_members = group_members; rp.group_offsets = group_offsets; rp.lite_mask = lite_mask;
  rp.K = group_size; rp.percentile = percentile;
  rp.group_fitness = group_fitness; rp.theta = theta; rp.route = route;
  sq::sq_route_kernel<<<(unsigned)num_problems, sq::ROUTE_THREADS, 0, static_cast<cudaStream_t>(stream)>>>(rp);
  ctx->launches += 1;
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
}

extern "C" int sq_score_select_prob(sq_score_ctx* ctx, const float* fitness, const int32_t* pop_offsets, int num_problems,
                                    float zeta, float* prob, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_problems < 0 || !(zeta > 0.f)) return set_err(ctx, SQ_ERR_INVALID_ARG, "num_problems >= 0 and zeta > 0 required");
  if (num_problems == 0) return SQ_OK;
  if (!fitness || !pop_offsets || !prob) return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  sq::SelectParams sp = {};
  sp.fitness = fitness; sp.pop_offsets = pop_offsets; sp.inv_zeta = 1.f / zeta; sp.prob = prob;
  sq::sq_select_prob_kernel<<<(unsigned)num_problems, sq::ROUTE_THREADS, 0, static_cast<cudaStream_t>(stream)>>>(sp);
  ctx->launches += 1;
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
}
