// sq_score_api.cu -- C ABI of libsq_score.so (include/sq_score.h): context, planning, TMA tensor
// maps and kernel launches.  No torch types, no CPU fallback.
#include "../../include/sq_score.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <queue>
#include <vector>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "sq_finalize_kernel.cuh"
#include "sq_fused_kernel.cuh"
#include "sq_positions_kernel.cuh"
#include "sq_prepare_kernel.cuh"
#include "sq_quant_kernel.cuh"
#include "sq_reduce_kernel.cuh"
#include "sq_route_kernel.cuh"

#define SQ_VERSION 200

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
  unsigned int* tail_counter = nullptr;   // CTAs of the finalize kernel that have finished (small runs; zero between runs)
  float* thr_pub = nullptr;   // [THR_MAX_CHUNKS][max_tokens] shared top-k bounds (sq_fused_kernel.cuh)
  // per-token scratch (used when the caller passes NULL per-token outputs)
  float* tok_lse = nullptr; float* tok_lp = nullptr; float* tok_ent = nullptr; float* tok_conf = nullptr;
  // kernel 2 workspace
  unsigned int* amax_bits = nullptr;   // per-tensor amax of sq_score_quantize_fp8
  int* seq_done = nullptr;   // [max_seqs] per-sequence tile counters of the single-launch reduction (zero between runs)
  int* tile_base = nullptr; int* tile_seq = nullptr; float4* red_sum = nullptr; float* red_min = nullptr; int64_t red_tiles_max = 0;
  int cluster4 = -1;                 // quad scheduling with W multicast (sq_fused_kernel.cuh): -1 = for very long runs only (default),
                                     // 0 = never, 1 = every run of more than 4096 tokens (cfg.clusTER4)
  int max_clusters[5] = {0, 0, 0, 0, 0};   // [cg]: clusters of kernel 1 the device holds at once (occupancy query at create)
  int region_mult = 0;               // region barrier of kernel 1: regions of region_mult x (a common multiple of the gang sizes) token tiles; < 0: off
  long long wait_limit = 0;          // cycles a device-side wait may last before kernel 1 traps (0 = for ever)
  int* pos_base = nullptr;           // [max_seqs + 1] packed start of every candidate (sq_score_positions)
  // staging for sq_score_run_host / sq_score_run_x (SQ_FLAG_STAGING)
  void* h_stage = nullptr; int32_t* tgt_stage = nullptr; int32_t* cu_stage = nullptr; float* seq_stage = nullptr;
  // sq_score_run_host streams H in on its own copy stream while kernel 1 runs: one flag per block of rows
  cudaStream_t copy_stream = nullptr; cudaEvent_t ev_fork = nullptr, ev_small = nullptr, ev_join = nullptr;
  unsigned int* h_flags = nullptr; unsigned int* one_host = nullptr;
  // driver entry point for tensor-map encoding
  void* encode_fn = nullptr;
  // optional per-kernel timing (sq_score_set_profiling): events around kernel 1, finalize
  // and kernel 2 of the last SQ_PROFILE_RING profiled runs
  int profiling = 0; int debug_flags = 0; int reduce_form = 0;
  // the four tensor maps of the last run (H, W, scale factors of H and of W): encoding one costs the host tens of
  // microseconds, which a decode-shaped run (0.1-0.2 ms on the device) cannot hide; a map depends only on the key below
  struct { int T = -1, k = 0, V = 0, tile_n = 0, d = 0; sq_score_plan_t pl; } plan_cache;   // the last run's plan (host time, as below)
  struct TmapSlot { const void* base = nullptr; int64_t rows = -1; int d = 0, box = 0, kind = -1; CUtensorMap map; } tmaps[4];
  int64_t ev_count = 0, ev_read = 0;   // runs recorded / runs already handed out by sq_score_profile_read
  cudaEvent_t (*ev)[4] = nullptr;      // [SQ_PROFILE_RING][4]
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
constexpr int HOST_FLAG_ROWS_MIN = 2048;   // sq_score_run_host: rows of H per arrival flag (doubled until a run needs at most ...
constexpr int HOST_FLAGS_PER_RUN = 256;    // ... this many flags)

static int topk_cap_for(int k) { return k <= 8 ? 8 : (k <= 20 ? 20 : 32); }
static inline int64_t cdiv64(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ------------------------------------------------------------------------------------------ plan
// Work decomposition.  The persistent clusters are split into gangs; gang i has s_i members
// (sizes differ by at most one, so that EVERY cluster the device holds is used: 74 = 2 x 13 + 4 x 12) and owns a
// stripe of the vocabulary, cut into `chunks_per_gang` chunks.  A gang walks the token tiles in batches of s_i
// (member j takes tile b * s_i + j) and sweeps its chunks for each batch, all members on the same W tile at the same
// time: a W tile is fetched from HBM once per batch and served to the other members from L2, and all gangs are on
// about the same token tiles at the same time, so the H strips in flight are ~max s_i.  Stripe widths are chosen so
// that every gang finishes together: a gang with more members needs fewer batches and gets a wider stripe.
static void split_stripes(int nv, int ng, const int* batches, int* width, int minw) {
  // minimise max_i batches[i] * width[i] subject to sum width = nv, width >= minw: proportional to 1 / batches, then the
  // left-over tiles one at a time to the gang whose finishing time grows least
  double inv = 0.0;
  for (int i = 0; i < ng; ++i) inv += 1.0 / batches[i];
  int used = 0;
  for (int i = 0; i < ng; ++i) {
    width[i] = std::max(minw, (int)std::floor(nv * (1.0 / batches[i]) / inv));
    used += width[i];
  }
  while (used > nv) {   // the floor of minw tiles per gang overshot: take from the gang that finishes last
    int w = -1;
    for (int i = 0; i < ng; ++i)
      if (width[i] > minw && (w < 0 || (int64_t)batches[i] * width[i] > (int64_t)batches[w] * width[w])) w = i;
    --width[w]; --used;
  }
  if (used < nv) {
    // (a heap: decode-shaped plans have ~150 gangs and ~150 left-over tiles, and the host time of a 0.1 ms run matters)
    typedef std::pair<int64_t, int> Key;   // (finishing time with one more tile, gang): the smallest, lowest gang first
    std::priority_queue<Key, std::vector<Key>, std::greater<Key>> heap;
    for (int i = 0; i < ng; ++i) heap.push(Key((int64_t)batches[i] * (width[i] + 1), i));
    while (used < nv) {
      const int w = heap.top().second;
      heap.pop();
      ++width[w]; ++used;
      heap.push(Key((int64_t)batches[w] * (width[w] + 1), w));
    }
  }
}

static int make_plan(const sq_score_config* cfg, int64_t T, int k, int num_sms, sq_score_plan_t* pl, int max_clusters = 0,
                     int tile_n = sq::BLOCK_N) {
  if (!cfg || !pl || T < 0 || cfg->d <= 0 || cfg->vocab <= 0 || k < 1 || k > SQ_MAX_K) return SQ_ERR_INVALID_ARG;
  if (num_sms <= 0) num_sms = 148;
  // default: CTA pairs (UMMA M = 256); a decode-shaped run of at most 128 rows fits one CTA's 128 TMEM
  // lanes, so single-CTA UMMA (M = 128) halves the wasted MMA rows and lets all 148 SMs stream W
  const int cg = (cfg->cta_group == 4) ? 4 : (cfg->cta_group == 1) ? 1 : (cfg->cta_group == 2 ? 2 : ((T > 0 && T <= 128) ? 1 : 2));
  memset(pl, 0, sizeof(*pl));
  pl->cta_group = cg;
  pl->rows_per_tile = 128 * cg;
  pl->m_tiles = (int)cdiv64(T, pl->rows_per_tile);
  pl->num_vtiles = (int)cdiv64(cfg->vocab, tile_n);   // 256 columns per tile (224 in the MX variant)
  pl->num_k_blocks = (int)cdiv64(cfg->d, 64);
  pl->num_clusters = std::max(1, num_sms / cg);
  if (max_clusters > 0) pl->num_clusters = std::min(pl->num_clusters, max_clusters);   // what can be co-resident (create)
  pl->topk_cap = topk_cap_for(k);
  const int M = std::max(1, pl->m_tiles), NV = pl->num_vtiles, NC = pl->num_clusters;
  const int gangs_max = std::min(NV, (int)sq::FIN_MAX_CHUNKS);   // every gang owns at least one vocab tile and one chunk

  // one candidate: `ng` gangs over min(NC, ng * M) clusters; cost in tile-times = the gang that finishes last
  struct Cand { int ng, base, big, r; double cost; };
  int batches[sq::FIN_MAX_CHUNKS], width[sq::FIN_MAX_CHUNKS];
  auto eval = [&](int ng, int r) {
    Cand c; c.ng = ng; c.r = r;
    c.base = std::min(NC / ng, M);                       // a member beyond the M-th would never get a token tile
    c.big = (c.base < M) ? std::min(NC - ng * c.base, ng) : 0;
    if (c.base + 1 > M) c.big = 0;
    for (int i = 0; i < ng; ++i) batches[i] = (int)cdiv64(M, c.base + (i < c.big ? 1 : 0));
    split_stripes(NV, ng, batches, width, r);
    double cost = 0.0;
    for (int i = 0; i < ng; ++i) cost = std::max(cost, batches[i] * (width[i] + 0.75 * std::min(r, width[i])));   // 0.75 tile of fill/drain per unit
    c.cost = cost;
    return c;
  };
  Cand best = {0, 0, 0, 1, 1e300};
  if (cfg->num_chunks > 0) {
    // forced number of chunks (tests, experiments): the largest gang count that divides it
    const int C = std::min(cfg->num_chunks, gangs_max);
    const int g_want = cfg->group_m > 0 ? cfg->group_m : 12;
    const int ng_hi = std::max(1, std::min(NC / std::max(1, std::min(g_want, std::min(M, NC))), C));
    int ng = 1;
    for (int n = 1; n <= ng_hi; ++n) if (C % n == 0) ng = n;
    best = eval(ng, C / ng);
  } else {
    // Gang size: 12 measured best on B200 at qwen3_8b / gpt_oss (swept 8 .. 36); neighbouring sizes are within
    // noise of one another, so the planner takes the size in 8 .. 16 whose batches and stripes quantise best for this T,
    // charging 1 % per step away from 12 (smaller gangs re-read W more often, larger ones keep more H strips in L2).
    double best_adj = 1e300;
    for (int dist = 0; dist <= (cfg->group_m > 0 ? 0 : 4); ++dist)
      for (int sgn = -1; sgn <= 1; sgn += 2) {
        if (dist == 0 && sgn > 0) continue;
        const int g = cfg->group_m > 0 ? cfg->group_m : 12 + sgn * dist;
        const int G = std::max(1, std::min(g, std::min(M, NC)));
        const int ng = std::max(1, std::min(NC / G, gangs_max));
        if (ng == best.ng) continue;                       // the same decomposition, further from the preferred gang size
        const Cand c = eval(ng, 1);
        const double adj = c.cost * (1.0 + 0.01 * dist);
        if (adj < best_adj * (1.0 - 1e-9)) { best_adj = adj; best = c; }
      }
    // Few token tiles (decode-shaped runs: the gang size is capped by M and clusters are to spare): every gang streams
    // its own stripe of W once and the run is HBM-bound, so all gangs should finish TOGETHER -- 594 tiles over 148 SMs
    // is 146 x 4 + 2 x 5, and the two 5-tile SMs would stream their last tile alone at a single SM's bandwidth (measured
    // +13 us on 197); 119 gangs x 5 tiles (118 x 5 + 4) finish together.  Take the fewest gangs with the same widest
    // stripe (also fewer partial states to merge).
    if (best.base == M && best.big == 0) {
      const int widest = (int)cdiv64(NV, best.ng);
      int ng = best.ng;
      while (ng > 1 && (int)cdiv64(NV, ng - 1) == widest) --ng;
      if (ng != best.ng) best = eval(ng, 1);
    }
  }
  pl->num_gangs = best.ng;
  pl->gang_size = best.base;
  pl->gangs_big = best.big;
  pl->chunks_per_gang = best.r;
  pl->num_chunks = best.ng * best.r;
  pl->clusters_used = best.ng * best.base + best.big;
  pl->num_units = pl->m_tiles * pl->num_chunks;
  for (int i = 0; i < best.ng; ++i) batches[i] = (int)cdiv64(M, best.base + (i < best.big ? 1 : 0));
  split_stripes(NV, best.ng, batches, width, best.r);
  // a gang's stripe is cut into r chunks of near-equal width (every stripe is at least r tiles wide: no empty chunk)
  int vt = 0, c = 0, widest = 0;
  pl->chunk_vtile[0] = 0;
  for (int i = 0; i < best.ng; ++i) {
    for (int q = 0; q < best.r; ++q) {
      const int w = width[i] / best.r + (q < width[i] % best.r ? 1 : 0);
      vt += w;
      widest = std::max(widest, w);
      pl->chunk_vtile[++c] = vt;
    }
    pl->max_batches = std::max(pl->max_batches, batches[i]);
  }
  pl->tiles_per_chunk = widest;
  if (pl->m_tiles == 0) pl->max_batches = 0;
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
extern "C" int sq_score_reduce_form(const sq_score_ctx* ctx) { return ctx ? ctx->reduce_form : 0; }
extern "C" int sq_score_last_plan(const sq_score_ctx* ctx, sq_score_plan_t* plan) {
  if (!ctx || !plan || ctx->plan_cache.T <= 0) return SQ_ERR_INVALID_ARG;
  *plan = ctx->plan_cache.pl;
  return SQ_OK;
}

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
  void* bufs[] = {ctx->tail_counter, ctx->amax_bits, ctx->seq_done, ctx->thr_pub, ctx->gang_ctr, ctx->part_cs, ctx->part_cu, ctx->part_m, ctx->part_s, ctx->part_u, ctx->part_topv, ctx->part_topi, ctx->zt,
                  ctx->tok_lse, ctx->tok_lp, ctx->tok_ent, ctx->tok_conf, ctx->tile_base, ctx->tile_seq, ctx->red_sum,
                  ctx->red_min, ctx->h_stage, ctx->tgt_stage, ctx->cu_stage, ctx->seq_stage, ctx->pos_base};
  int rc = SQ_OK;
  for (void* b : bufs)
    if (b && cudaFree(b) != cudaSuccess) rc = SQ_ERR_CUDA;
  if (ctx->ev) {
    for (int i = 0; i < SQ_PROFILE_RING; ++i)
      for (cudaEvent_t e : ctx->ev[i])
        if (e) cudaEventDestroy(e);
    delete[] ctx->ev;
  }
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
  if (cfg->cta_group < 0 || cfg->cta_group > 2 || cfg->num_chunks < 0 || cfg->group_m < 0 ||
      (cfg->flags & ~(SQ_FLAG_REDUCE_ONLY | SQ_FLAG_STAGING)) || (cfg->debug_flags & ~SQ_DEBUG_ALL) || cfg->region_mult < -1)
    return set_err(nullptr, SQ_ERR_INVALID_ARG, "cta_group must be 0, 1 or 2; num_chunks, group_m >= 0; region_mult >= -1; unknown flag");
  if (cfg->vocab > SQ_MAX_VOCAB)   // 65535 tiles of the narrowest tile width (224 columns, MX variant)
    return set_err(nullptr, SQ_ERR_UNSUPPORTED, "vocab = %d exceeds %d (vocab-tile indices are 16-bit: at most 65535 tiles of 224 columns)",
                   cfg->vocab, SQ_MAX_VOCAB);
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
  ctx->cap_max = topk_cap_for(cfg->max_k);
  // cfg.debug_flags selects between code paths that give the SAME results (tests force each of them): bit 3 = two-pass
  // prepare kernel, bit 4 = no shared top-k bound, bit 5 / 6 = three-launch / single-launch kernel 2, bit 7 = one warp
  // per row in the finalize kernel
  ctx->debug_flags = cfg->debug_flags;
  ctx->region_mult = cfg->region_mult;                                  // 0 = default, > 0 forced, -1 = no region barrier
  ctx->cluster4 = cfg->cluster4 == 0 ? -1 : (cfg->cluster4 > 0 ? 1 : 0);   // -1 = long runs only (default), 1 = always, 0 = never
  {   // device-side waits trap after cfg.wait_seconds (default 60 s; raise it under a sanitizer)
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, cfg->device);
    long long sec = cfg->wait_seconds == 0 ? 60 : cfg->wait_seconds;
    sec = std::min<long long>(sec, 1000000000LL);   // keeps the cycle count far inside 63 bits (31 years are for ever too)
    ctx->wait_limit = sec < 0 ? 0 : sec * (long long)std::max(khz, 1000000) * 1000LL;
  }

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
  // kernel 2's partial records: tile forms (one per 8192-token tile) or streaming form (one per 256-token range and sequence)
  ctx->red_tiles_max = std::max<int64_t>(cdiv64(T, sq::RED_TILE) + 2 * (int64_t)cfg->max_seqs + 1,
                                         2 * cdiv64(T, sq::RsCfg<2>::TB) * sq::RS_WARPS + 2);   // (red_min: two floats per range; the smaller ranges)
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
  A(ws_alloc(ctx, &ctx->tail_counter, 1));
  if (rc == SQ_OK && cudaMemset(ctx->tail_counter, 0, sizeof(unsigned int)) != cudaSuccess) rc = SQ_ERR_CUDA;
  A(ws_alloc(ctx, &ctx->seq_done, (int64_t)cfg->max_seqs));
  if (rc == SQ_OK && cudaMemset(ctx->seq_done, 0, (size_t)cfg->max_seqs * sizeof(int)) != cudaSuccess) rc = SQ_ERR_CUDA;
  A(ws_alloc(ctx, &ctx->red_sum, ctx->red_tiles_max));
  A(ws_alloc(ctx, &ctx->tile_seq, ctx->red_tiles_max));
  A(ws_alloc(ctx, &ctx->red_min, ctx->red_tiles_max));
  A(ws_alloc(ctx, &ctx->seq_stage, 4 * (int64_t)cfg->max_seqs));
  A(ws_alloc(ctx, &ctx->pos_base, (int64_t)cfg->max_seqs + 1));
  if ((cfg->flags & SQ_FLAG_STAGING) && !reduce_only) {   // everything sq_score_run_host / sq_score_run_x need: no run allocates
    A(ws_alloc(ctx, reinterpret_cast<uint8_t**>(&ctx->h_stage), T * (int64_t)cfg->d * 2));
    A(ws_alloc(ctx, &ctx->tgt_stage, T));
    A(ws_alloc(ctx, &ctx->cu_stage, (int64_t)cfg->max_seqs + 1));
    A(ws_alloc(ctx, &ctx->h_flags, HOST_FLAGS_PER_RUN));
    if (rc == SQ_OK) {
      bool ok = cudaHostAlloc(reinterpret_cast<void**>(&ctx->one_host), sizeof(unsigned int), cudaHostAllocDefault) == cudaSuccess;
      if (ok) *ctx->one_host = 1u;
      ok = ok && cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) == cudaSuccess;
      ok = ok && cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) == cudaSuccess;
      ok = ok && cudaEventCreateWithFlags(&ctx->ev_small, cudaEventDisableTiming) == cudaSuccess;
      ok = ok && cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) == cudaSuccess;
      if (!ok) { rc = SQ_ERR_CUDA; set_err(ctx, rc, "creating the copy stream / events failed: %s", cudaGetErrorString(cudaGetLastError())); }
    }
  }
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
#define SQ_SET_SMEM8(CG, CAP)                                                                                              \
  if (cudaFuncSetAttribute(sq::sq_fused_score_kernel<CG, CAP, sq::MODE_F8>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                           sq::FusedCfg<CG, sq::MODE_F8>::SMEM_BYTES) != cudaSuccess) rc = SQ_ERR_CUDA;                    \
  if (cudaFuncSetAttribute(sq::sq_fused_score_kernel<CG, CAP, sq::MODE_MX>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                           sq::FusedCfg<CG, sq::MODE_MX>::SMEM_BYTES) != cudaSuccess) rc = SQ_ERR_CUDA;
  SQ_SET_SMEM8(1, 8) SQ_SET_SMEM8(1, 20) SQ_SET_SMEM8(1, 32) SQ_SET_SMEM8(2, 8) SQ_SET_SMEM8(2, 20) SQ_SET_SMEM8(2, 32)
#undef SQ_SET_SMEM8
#define SQ_SET_SMEM_H(CAP, MODE)                                                                                                 \
  if (cudaFuncSetAttribute(sq::sq_fused_score_kernel<1, CAP, MODE, 1, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize,         \
                           sq::FusedCfg<1, MODE, 64>::SMEM_BYTES) != cudaSuccess) rc = SQ_ERR_CUDA;                              \
  if (cudaFuncSetAttribute(sq::sq_fused_score_kernel<1, CAP, MODE, 1, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize,         \
                           sq::FusedCfg<1, MODE, 32>::SMEM_BYTES) != cudaSuccess) rc = SQ_ERR_CUDA;
  SQ_SET_SMEM_H(8, sq::MODE_BF16) SQ_SET_SMEM_H(20, sq::MODE_BF16) SQ_SET_SMEM_H(32, sq::MODE_BF16)
  SQ_SET_SMEM_H(8, sq::MODE_F8) SQ_SET_SMEM_H(20, sq::MODE_F8) SQ_SET_SMEM_H(32, sq::MODE_F8)
  SQ_SET_SMEM_H(8, sq::MODE_MX) SQ_SET_SMEM_H(20, sq::MODE_MX) SQ_SET_SMEM_H(32, sq::MODE_MX)
#undef SQ_SET_SMEM_H
  for (const void* f : {(const void*)sq::sq_fused_score_kernel<2, 8, sq::MODE_BF16, 4>, (const void*)sq::sq_fused_score_kernel<2, 20, sq::MODE_BF16, 4>,
                        (const void*)sq::sq_fused_score_kernel<2, 32, sq::MODE_BF16, 4>, (const void*)sq::sq_fused_score_kernel<2, 8, sq::MODE_F8, 4>,
                        (const void*)sq::sq_fused_score_kernel<2, 20, sq::MODE_F8, 4>, (const void*)sq::sq_fused_score_kernel<2, 32, sq::MODE_F8, 4>})
    if (cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, sq::FusedCfg<2>::SMEM_BYTES) != cudaSuccess) rc = SQ_ERR_CUDA;
  for (const void* f : {(const void*)sq::sq_reduce_fused_kernel<true>, (const void*)sq::sq_reduce_fused_kernel<false>})
    if (cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             sq::RED_SMEM_BYTES + (sq::RED_FUSED_MAX_SEQS + 1) * (int)sizeof(int)) != cudaSuccess) rc = SQ_ERR_CUDA;
  if (rc != SQ_OK) {
    set_err(nullptr, rc, "cudaFuncSetAttribute(MaxDynamicSharedMemorySize) failed: %s", cudaGetErrorString(cudaGetLastError()));
    sq_score_destroy(ctx);
    return rc;
  }
  // Kernel 1's clusters wait for one another (gang barriers), so all of them must be resident at once: ask the
  // occupancy calculator how many the device holds (it knows the shared-memory footprint, the cluster shape and any
  // SM partitioning of this context) and plan for at most that many.
  if (!reduce_only) {
    for (int cg = 1; cg <= 2; ++cg) {
      cudaLaunchConfig_t lc = {};
      lc.gridDim = dim3((unsigned)(ctx->num_sms / cg * cg));
      lc.blockDim = dim3(sq::NUM_THREADS);
      lc.dynamicSmemBytes = cg == 1 ? sq::FusedCfg<1>::SMEM_BYTES : sq::FusedCfg<2>::SMEM_BYTES;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = cg; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      lc.attrs = at; lc.numAttrs = 1;
      int n = 0;
      const cudaError_t oe = cg == 1 ? cudaOccupancyMaxActiveClusters(&n, sq::sq_fused_score_kernel<1, 32>, &lc)
                                     : cudaOccupancyMaxActiveClusters(&n, sq::sq_fused_score_kernel<2, 32>, &lc);
      if (oe != cudaSuccess || n < 1) {
        set_err(nullptr, SQ_ERR_UNSUPPORTED, "the device cannot hold a cluster of %d CTA(s) of the fused kernel (%s)", cg,
                oe == cudaSuccess ? "occupancy 0" : cudaGetErrorString(oe));
        cudaGetLastError();
        sq_score_destroy(ctx);
        return SQ_ERR_UNSUPPORTED;
      }
      ctx->max_clusters[cg] = n;
    }
    if (ctx->cluster4) ctx->max_clusters[4] = ctx->max_clusters[2] / 2;   // quads: 4 consecutive CTAs, placed as one cluster of 4 or two of 2
    if (ctx->max_clusters[4] * 4 != ctx->num_sms / 4 * 4) ctx->max_clusters[4] = 0;   // (only when every quad fits at once)
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
static int make_tmap(sq_score_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int d, int box_rows, bool f8 = false, int slot = -1) {
  if (slot >= 0) {
    const sq_score_ctx::TmapSlot& c = ctx->tmaps[slot];
    if (c.base == base && c.rows == rows && c.d == d && c.box == box_rows && c.kind == (f8 ? 1 : 0)) { *map = c.map; return SQ_OK; }
  }
  const cuuint64_t dims[2] = {(cuuint64_t)d, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)d * (f8 ? 1 : 2)};
  const cuuint32_t box[2] = {(cuuint32_t)(f8 ? sq::BLOCK_K_F8 : sq::BLOCK_K), (cuuint32_t)box_rows};   // 128 bytes wide
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = reinterpret_cast<encode_tiled_fn>(ctx->encode_fn)(
      map, f8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_err(ctx, SQ_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  if (slot >= 0) {
    sq_score_ctx::TmapSlot& c = ctx->tmaps[slot];
    c.base = base; c.rows = rows; c.d = d; c.box = box_rows; c.kind = f8 ? 1 : 0; c.map = *map;
  }
  return SQ_OK;
}

// MX scale factors: `rows` rows of 512 bytes (128 x uint32), unswizzled; a box is `box_rows` whole rows.
static int make_tmap_sf(sq_score_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int box_rows, int slot) {
  {
    const sq_score_ctx::TmapSlot& c = ctx->tmaps[slot];
    if (c.base == base && c.rows == rows && c.box == box_rows && c.kind == 2) { *map = c.map; return SQ_OK; }
  }
  const cuuint64_t dims[2] = {128, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {512};
  const cuuint32_t box[2] = {128, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = reinterpret_cast<encode_tiled_fn>(ctx->encode_fn)(
      map, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(base), dims, strides, box, estr,
      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_err(ctx, SQ_ERR_CUDA, "cuTensorMapEncodeTiled (scale factors) failed with CUresult %d", (int)r);
  sq_score_ctx::TmapSlot& c = ctx->tmaps[slot];
  c.base = base; c.rows = rows; c.d = 0; c.box = box_rows; c.kind = 2; c.map = *map;
  return SQ_OK;
}

// ------------------------------------------------------------------------------------------ launches
template <int CG, int CAP, int MODE = sq::MODE_BF16, int CL = CG, int AROWS = 128>
static cudaError_t launch_fused(const sq_score_plan_t& pl, int num_sms, const CUtensorMap& th, const CUtensorMap& tw,
                                const CUtensorMap& tsa, const CUtensorMap& tsb, const sq::FusedParams& fp, cudaStream_t st) {
  const int clusters = pl.clusters_used;   // every launched cluster belongs to a gang
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)(clusters * CL));
  lc.blockDim = dim3(sq::NUM_THREADS);
  lc.dynamicSmemBytes = sq::FusedCfg<CG, MODE, AROWS>::SMEM_BYTES;
  lc.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = CG; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  lc.attrs = at;
  lc.numAttrs = 1;
  if (CL == 4) {   // quads: clusters of 4 where the device can place them, pairs elsewhere (sq_fused_kernel.cuh)
    at[1].id = cudaLaunchAttributePreferredClusterDimension;
    at[1].val.preferredClusterDim.x = 4; at[1].val.preferredClusterDim.y = 1; at[1].val.preferredClusterDim.z = 1;
    lc.numAttrs = 2;
  }
  (void)num_sms;
  return cudaLaunchKernelEx(&lc, sq::sq_fused_score_kernel<CG, CAP, MODE, CL, AROWS>, th, tw, tsa, tsb, fp);
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

// rows swept by more than 32 vocab chunks: one CTA per row (sq_finalize_wide_kernel), compiled per list capacity
template <bool EMIT>
static cudaError_t launch_wide_finalize(int cap, int T, cudaStream_t st, const sq::FinalizeParams& fin) {
  const dim3 grid((unsigned)T), block(sq::FIN_WIDE_THREADS);
  if (cap == 8) return launch_pdl(sq::sq_finalize_wide_kernel<8, EMIT>, grid, block, 0, st, fin);
  if (cap == 20) return launch_pdl(sq::sq_finalize_wide_kernel<20, EMIT>, grid, block, 0, st, fin);
  return launch_pdl(sq::sq_finalize_wide_kernel<32, EMIT>, grid, block, 0, st, fin);
}

#ifndef SQ_RS_NV_NOTG
#define SQ_RS_NV_NOTG 3
#endif
static int launch_reduce(sq_score_ctx* ctx, sq::ReduceParams& rp, cudaStream_t st) {
  if (rp.B <= 0) return SQ_OK;
  // 16-byte loads need 16-byte aligned arrays (tiles start on multiples of 4 tokens)
  rp.vec = ((((uintptr_t)rp.lp | (uintptr_t)rp.ent | (uintptr_t)rp.conf | (uintptr_t)rp.targets) & 15) == 0) ? 1 : 0;
  const int64_t tiles = cdiv64(rp.T, sq::RED_TILE) + 2 * (int64_t)rp.B;   // upper bound on sum_b ceil((L_b + 3) / RED_TILE)
  // Single launch (sq_reduce_kernel.cuh) when the whole problem is one wave of CTAs -- the scoring pipeline's case, a few
  // dozen tiles, where the three launches are pure latency (20 -> 8 us).  On large inputs the three-launch form is 2x
  // faster (measured 0.099 vs 0.218 ms on 3.6e7 tokens: a persistent CTA pays the fence + atomic + barriers per tile in
  // series), so it stays.  cfg.debug_flags bit 5 / bit 6 force the three-launch / single-launch form (tests).
  const size_t fused_smem = sq::RED_SMEM_BYTES + (size_t)(rp.B + 1) * sizeof(int);
  const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(6, (size_t)(220 * 1024) / (fused_smem + 1024)));
  const bool one_wave = tiles <= (int64_t)ctx->num_sms * per_sm && rp.B <= 2048;
  if (rp.B <= sq::RED_FUSED_MAX_SEQS && !(ctx->debug_flags & (32 | 256)) && (one_wave || (ctx->debug_flags & 64))) {
    rp.seq_done = ctx->seq_done;
    const size_t smem = fused_smem;
    const dim3 grid((unsigned)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)ctx->num_sms * per_sm)));
    if (rp.targets) SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_fused_kernel<true>, grid, dim3(sq::RED_THREADS), smem, st, rp));
    else SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_fused_kernel<false>, grid, dim3(sq::RED_THREADS), smem, st, rp));
    ctx->launches += 1;
    ctx->reduce_form = SQ_REDUCE_FORM_FUSED;
    SQ_CUDA(ctx, cudaGetLastError());
    return SQ_OK;
  }
  // Streaming form (two launches, sq_reduce_kernel.cuh): fixed 4096-token blocks whose loads depend on nothing, every
  // sequence boundary handled in the fold.  Needs 16-byte aligned arrays and RS_WMIN <= window <= RS_WMAX; cfg.debug_flags bit 8 forces
  // it on small inputs (tests).
  // Narrow windows stay with the tile forms: the streaming form takes S(j) as a difference of two block-wide prefix sums,
  // whose fp32 rounding (~1e-7 of the prefix) is only negligible against a sum of >= RS_WMIN elements.
  if (rp.vec && rp.window >= sq::RS_WMIN && rp.window <= sq::RS_WMAX && rp.T > 0 &&
      rp.T <= (int64_t)INT32_MAX - 2 * (sq::RsCfg<3>::TB + sq::RS_WMAX) &&
      !(ctx->debug_flags & (32 | 64))) {
    const dim3 fgrid((unsigned)cdiv64(rp.B, 4));
    if (rp.targets) {   // four arrays: two vectors per lane and array; three arrays: three (sq_reduce_kernel.cuh)
      SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_stream_kernel<true, 2>, dim3((unsigned)cdiv64(rp.T, sq::RsCfg<2>::TB)), dim3(sq::RS_THREADS), 0, st, rp));
      SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_stream_fold_kernel<2>, fgrid, dim3(128), 0, st, rp));
    } else {
      SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_stream_kernel<false, SQ_RS_NV_NOTG>, dim3((unsigned)cdiv64(rp.T, sq::RsCfg<SQ_RS_NV_NOTG>::TB)), dim3(sq::RS_THREADS), 0, st, rp));
      SQ_CUDA(ctx, launch_pdl(sq::sq_reduce_stream_fold_kernel<SQ_RS_NV_NOTG>, fgrid, dim3(128), 0, st, rp));
    }
    ctx->launches += 2;
    ctx->reduce_form = SQ_REDUCE_FORM_STREAM;
    SQ_CUDA(ctx, cudaGetLastError());
    return SQ_OK;
  }
  ctx->reduce_form = SQ_REDUCE_FORM_TILES;
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

// ------------------------------------------------------------------------------------------ kernel 2 without a ctx
// sq_score_reduce_static (include/sq_score.h): kernel 2's single-launch form for callers that must not allocate.  What
// a ctx keeps in cudaMalloc'ed workspace -- one float4 + one float per tile, one counter per sequence -- lives in the
// array below, which is part of the library's device image: the driver places it when the module is loaded on a device
// and it stays until the process exits.  Sized for the stated maxima (tiles <= ceil(T / RED_TILE) + 2 B).
constexpr int64_t STATIC_MAX_TILES = (SQ_STATIC_MAX_TOKENS + sq::RED_TILE - 1) / sq::RED_TILE + 2 * (int64_t)SQ_STATIC_MAX_SEQS;
constexpr size_t STATIC_OFF_SUM = 0;                                                                  // float4 [tiles]
constexpr size_t STATIC_OFF_MIN = (STATIC_OFF_SUM + STATIC_MAX_TILES * sizeof(float4) + 255) / 256 * 256;   // float [tiles]
constexpr size_t STATIC_OFF_DONE = (STATIC_OFF_MIN + STATIC_MAX_TILES * sizeof(float) + 255) / 256 * 256;   // int [seqs]
constexpr size_t STATIC_BYTES = (STATIC_OFF_DONE + SQ_STATIC_MAX_SEQS * sizeof(int) + 255) / 256 * 256;
static_assert(SQ_STATIC_MAX_SEQS <= sq::RED_FUSED_MAX_SEQS, "the single-launch form keeps B + 1 ints in shared memory");
static_assert(STATIC_BYTES <= 256 * 1024, "keep the resident scratch modest: every GPU that loads the library holds it");

static __device__ __align__(256) unsigned char g_static_scratch[STATIC_BYTES];

// In host code `g_static_scratch` is only a handle for the runtime's symbol table, not a device address: the address a
// kernel may use comes from cudaGetSymbolAddress, per device (every device has its own copy of the array).
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDev { unsigned char* base; int num_sms; };
static StaticDev g_static_dev[STATIC_MAX_DEVICES] = {};
static std::mutex g_static_mu;

// Set-up of the calling thread's current device `dev`, once: host-side queries only, nothing is allocated.
static int static_setup(int dev, StaticDev* out) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_dev[dev].base) {
    int major = 0, sms = 0;
    SQ_CUDA(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10)
      return set_err(nullptr, SQ_ERR_CUDA, "device %d is sm_%dx; the kernels are built for sm_100a only", dev, major);
    SQ_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    unsigned char* base = nullptr;
    SQ_CUDA(nullptr, cudaGetSymbolAddress(reinterpret_cast<void**>(&base), g_static_scratch));
    if (!base || ((uintptr_t)base & 255)) return set_err(nullptr, SQ_ERR_CUDA, "cudaGetSymbolAddress gave %p for the scratch array", (void*)base);
    // the same limit sq_score_create sets (it is per kernel and device, shared with every ctx: never a smaller one)
    for (const void* f : {(const void*)sq::sq_reduce_fused_kernel<true>, (const void*)sq::sq_reduce_fused_kernel<false>})
      SQ_CUDA(nullptr, cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            sq::RED_SMEM_BYTES + (sq::RED_FUSED_MAX_SEQS + 1) * (int)sizeof(int)));
    g_static_dev[dev].num_sms = sms;
    g_static_dev[dev].base = base;
  }
  *out = g_static_dev[dev];
  return SQ_OK;
}

extern "C" int sq_score_reduce_static(const float* target_logprob, const float* entropy, const float* conf,
                                      const int32_t* targets, const int32_t* cu_seqlens, int64_t num_tokens, int num_seqs,
                                      int vocab, int window, float* seq_mean_logprob, float* seq_mean_entropy,
                                      float* seq_mean_conf, float* seq_min_window_conf, void* stream) {
  if (num_tokens < 0 || num_seqs < 0 || window < 1)
    return set_err(nullptr, SQ_ERR_INVALID_ARG, "sq_score_reduce_static: T, B >= 0 and window >= 1 required");
  if (num_tokens > SQ_STATIC_MAX_TOKENS || num_seqs > SQ_STATIC_MAX_SEQS)
    return set_err(nullptr, SQ_ERR_INVALID_ARG,
                   "sq_score_reduce_static: T = %lld / B = %d exceed the fixed scratch (at most %d tokens and %d sequences per "
                   "call); larger inputs need sq_score_create + sq_score_reduce",
                   (long long)num_tokens, num_seqs, SQ_STATIC_MAX_TOKENS, SQ_STATIC_MAX_SEQS);
  if (num_seqs == 0) return SQ_OK;
  if (!cu_seqlens || !seq_mean_logprob || !seq_mean_entropy || !seq_mean_conf || !seq_min_window_conf ||
      (num_tokens > 0 && (!target_logprob || !entropy || !conf)))
    return set_err(nullptr, SQ_ERR_INVALID_ARG, "sq_score_reduce_static: null pointer argument");
  if (targets && vocab < 1) return set_err(nullptr, SQ_ERR_INVALID_ARG, "sq_score_reduce_static: vocab >= 1 required with targets");
  int dev = -1;
  SQ_CUDA(nullptr, cudaGetDevice(&dev));
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return set_err(nullptr, SQ_ERR_CUDA, "sq_score_reduce_static: device ordinal %d not supported", dev);
  StaticDev sd;
  const int rc = static_setup(dev, &sd);
  if (rc != SQ_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  sq::ReduceParams rp = {};
  rp.T = num_tokens; rp.B = num_seqs; rp.V = targets ? vocab : 1; rp.window = window;
  rp.lp = target_logprob; rp.ent = entropy; rp.conf = conf; rp.targets = targets; rp.cu = cu_seqlens;
  rp.part_sum = reinterpret_cast<float4*>(sd.base + STATIC_OFF_SUM);
  rp.part_min = reinterpret_cast<float*>(sd.base + STATIC_OFF_MIN);
  rp.seq_done = reinterpret_cast<int*>(sd.base + STATIC_OFF_DONE);
  rp.out_lp = seq_mean_logprob; rp.out_ent = seq_mean_entropy; rp.out_conf = seq_mean_conf; rp.out_min = seq_min_window_conf;
  rp.vec = ((((uintptr_t)rp.lp | (uintptr_t)rp.ent | (uintptr_t)rp.conf | (uintptr_t)rp.targets) & 15) == 0) ? 1 : 0;
  // the array keeps the last call's contents: the counters must be zero when the kernel starts
  SQ_CUDA(nullptr, cudaMemsetAsync(rp.seq_done, 0, (size_t)num_seqs * sizeof(int), st));
  const int64_t tiles = cdiv64(num_tokens, sq::RED_TILE) + 2 * (int64_t)num_seqs;   // <= STATIC_MAX_TILES by the size check
  const size_t smem = sq::RED_SMEM_BYTES + (size_t)(num_seqs + 1) * sizeof(int);
  const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(6, (size_t)(220 * 1024) / (smem + 1024)));
  const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)sd.num_sms * per_sm));
  // a plain launch behind the memset (no programmatic serialization: cudaGridDependencySynchronize() is then a no-op)
  if (targets) sq::sq_reduce_fused_kernel<true><<<grid, sq::RED_THREADS, smem, st>>>(rp);
  else sq::sq_reduce_fused_kernel<false><<<grid, sq::RED_THREADS, smem, st>>>(rp);
  SQ_CUDA(nullptr, cudaGetLastError());
  return SQ_OK;
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
                    const float* w_scale = nullptr, int shard_rows = 0, const void* h_sf = nullptr, const void* w_sf = nullptr) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (!o && !shard_state) return set_err(ctx, SQ_ERR_INVALID_ARG, "outputs is null");
  static const sq_score_outputs no_outputs = {};
  if (!o) o = &no_outputs;
  if (ctx->cfg.flags & SQ_FLAG_REDUCE_ONLY) return set_err(ctx, SQ_ERR_INVALID_ARG, "ctx was created with SQ_FLAG_REDUCE_ONLY");
  const int T = num_tokens, d = ctx->cfg.d;
  const int V = shard_state ? shard_rows : ctx->cfg.vocab;   // a vocab-parallel shard may hold fewer rows than the ctx was sized for
  int B = num_seqs;
  if (T < 0 || B < 0) return set_err(ctx, SQ_ERR_INVALID_ARG, "negative T or B");
  if (V < 1 || V > ctx->cfg.vocab) return set_err(ctx, SQ_ERR_INVALID_ARG, "shard_rows = %d outside 1..cfg.vocab = %d", V, ctx->cfg.vocab);
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
    const bool mx = h_sf != nullptr;                       // block-scaled e4m3 (sq_score_run_mx)
    const bool f8 = h_scale != nullptr || mx;              // 8-bit operands: 128 elements per k-block
    const int tile_n = mx ? sq::BLOCK_N_MX : sq::BLOCK_N;
    sq_score_plan_t pl;
    sq_score_config pc = ctx->cfg;
    pc.vocab = V;
    if (f8) pc.d = (d + 1) / 2;   // an e4m3 k-block is 128 elements: the plan sees half as many k-blocks
    int cg_sel = (pc.cta_group == 1) ? 1 : (pc.cta_group == 2 ? 2 : (T <= 128 ? 1 : 2));
    // Quads pay where kernel 1's energy goes into operand traffic for long: measured +2.4 % at qwen3_32b (T = 5e5), +1.2 % at
    // gpt_oss, +0.3 % (noise) at qwen3_8b, so by default only runs of more than 200 000 tokens take them.
    const int quad_min_t = ctx->cluster4 > 0 ? 4096 : 200000;
    if (ctx->cluster4 != 0 && cg_sel == 2 && !mx && pc.cta_group == 0 && T > quad_min_t && ctx->max_clusters[4] > 0) {
      cg_sel = 4; pc.cta_group = 4;
      if (pc.group_m == 0) pc.group_m = 6;             // gangs of 6 quads = 12 strips of 256 rows, the pair kernel's optimum
    }
    auto& pcache = ctx->plan_cache;
    if (pcache.T == T && pcache.k == k && pcache.V == V && pcache.tile_n == tile_n && pcache.d == pc.d) {
      pl = pcache.pl;
    } else {
      make_plan(&pc, T, k, ctx->num_sms, &pl, ctx->max_clusters[cg_sel], tile_n);
      const int64_t rows = ws_rows_for(ctx->cfg);
      if ((int64_t)pl.num_chunks * T > rows) {   // workspace bound: fewer gangs, wider stripes
        pc.num_chunks = (int)std::max<int64_t>(1, rows / T);
        make_plan(&pc, T, k, ctx->num_sms, &pl, ctx->max_clusters[cg_sel], tile_n);
      }
      pcache.T = T; pcache.k = k; pcache.V = V; pcache.tile_n = tile_n; pcache.d = pc.d; pcache.pl = pl;
    }
    if (pl.topk_cap > ctx->cap_max) return set_err(ctx, SQ_ERR_INVALID_ARG, "k exceeds the ctx's max_k capacity");
    if (pl.num_vtiles > 65535)   // FusedParams::chunk_vt is 16-bit: the last chunk's end would wrap to 0 and the chunk be skipped
      return set_err(ctx, SQ_ERR_UNSUPPORTED, "%d vocab tiles of %d columns exceed the 16-bit tile index", pl.num_vtiles, tile_n);
    CUtensorMap th, tw, tsa, tsb;
    if (f8 && d % 16 != 0) return set_err(ctx, SQ_ERR_UNSUPPORTED, "the FP8 variants need d %% 16 == 0 (TMA 16-byte row strides)");
    // decode-shaped, at most 64 / 32 rows: 64- / 32-row H boxes, five / six stages
    const int a_rows = (pl.cta_group == 1 && T <= 32) ? 32 : ((pl.cta_group == 1 && T <= 64) ? 64 : sq::BLOCK_M);
    int h_box = a_rows, w_box = tile_n / pl.cta_group;
    int rc = make_tmap(ctx, &th, H, T, d, h_box, f8, 0);
    if (rc != SQ_OK) return rc;
    rc = make_tmap(ctx, &tw, W, V, d, w_box, f8, 1);
    if (rc != SQ_OK) return rc;
    tsa = th; tsb = tw;                                    // unused outside the MX variant
    const int64_t sf_h_blocks = cdiv64(T, sq::BLOCK_M);
    if (mx) {   // rows of 512 scale bytes: [k-block][128-row block of H], [k-block][vocab tile][2]  (sq_quant_mx_kernel)
      rc = make_tmap_sf(ctx, &tsa, h_sf, (int64_t)pl.num_k_blocks * sf_h_blocks, 1, 2);
      if (rc != SQ_OK) return rc;
      rc = make_tmap_sf(ctx, &tsb, w_sf, (int64_t)pl.num_k_blocks * pl.num_vtiles * 2, 2, 3);
      if (rc != SQ_OK) return rc;
    }

    sq::FusedParams fp = {};
    fp.T = T; fp.V = V; fp.d = d;
    fp.num_k_blocks = pl.num_k_blocks; fp.num_vtiles = pl.num_vtiles;
    fp.num_chunks = pl.num_chunks; fp.m_tiles = pl.m_tiles;
    fp.num_gangs = pl.num_gangs; fp.gang_size = pl.gang_size; fp.gangs_big = pl.gangs_big;
    fp.chunks_per_gang = pl.chunks_per_gang; fp.gang_ctr = ctx->gang_ctr;
    fp.wait_limit = ctx->wait_limit;
    // region barrier (sq_fused_kernel.cuh): a region is a number of token tiles that every gang covers in whole batches
    fp.region_ctr = ctx->gang_ctr + 255; fp.region_tiles = 0; fp.region_arrivals = pl.clusters_used * pl.cta_group;
    if (pl.num_gangs > 1 && pl.gang_size + (pl.gangs_big > 0 ? 1 : 0) > 1) {
      const int unit = pl.gangs_big > 0 && pl.gangs_big < pl.num_gangs ? pl.gang_size * (pl.gang_size + 1) : pl.gang_size + (pl.gangs_big > 0 ? 1 : 0);
      const int mult = ctx->region_mult > 0 ? ctx->region_mult : std::max(1, 160 / unit);   // default: regions of ~160 token tiles
      if (ctx->region_mult >= 0 && unit * mult < pl.m_tiles) fp.region_tiles = unit * mult;
    }
    for (int c = 0; c <= pl.num_chunks; ++c) fp.chunk_vt[c] = (uint16_t)pl.chunk_vtile[c];
    // the gang barrier counters only matter when some gang has more than one member (not in decode-shaped plans)
    if (pl.gang_size + (pl.gangs_big > 0 ? 1 : 0) > 1)
      SQ_CUDA(ctx, cudaMemsetAsync(ctx->gang_ctr, 0, 256 * sizeof(unsigned int), st));
    fp.targets = targets;
    fp.part_m = ctx->part_m; fp.part_s = ctx->part_s; fp.part_u = ctx->part_u;
    fp.part_cs = ctx->part_cs; fp.part_cu = ctx->part_cu;
    fp.part_topv = ctx->part_topv; fp.part_topi = ctx->part_topi; fp.zt = ctx->zt;
    fp.vocab_offset = vocab_offset;
    fp.h_scale = h_scale; fp.w_scale = w_scale; fp.sf_h_blocks = (int)sf_h_blocks;
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
    cudaEvent_t* pev = ctx->profiling ? ctx->ev[ctx->ev_count % SQ_PROFILE_RING] : nullptr;
    if (pev) cudaEventRecord(pev[0], st);
    const int sel = pl.cta_group * 100 + pl.topk_cap + (mx ? 2000 : (f8 ? 1000 : 0)) + (a_rows == 64 ? 10000 : (a_rows == 32 ? 20000 : 0));
#define SQ_LAUNCH(CG, CAP, MODE) e = launch_fused<CG, CAP, MODE>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break
    switch (sel) {
#define SQ_LAUNCH_Q(CAP, MODE) e = launch_fused<1, CAP, MODE, 1, 32>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break
      case 22108: SQ_LAUNCH_Q(8, sq::MODE_MX);
      case 22120: SQ_LAUNCH_Q(20, sq::MODE_MX);
      case 22132: SQ_LAUNCH_Q(32, sq::MODE_MX);
      case 21108: SQ_LAUNCH_Q(8, sq::MODE_F8);
      case 21120: SQ_LAUNCH_Q(20, sq::MODE_F8);
      case 21132: SQ_LAUNCH_Q(32, sq::MODE_F8);
      case 20108: SQ_LAUNCH_Q(8, sq::MODE_BF16);
      case 20120: SQ_LAUNCH_Q(20, sq::MODE_BF16);
      case 20132: SQ_LAUNCH_Q(32, sq::MODE_BF16);
#undef SQ_LAUNCH_Q
#define SQ_LAUNCH_H(CAP, MODE) e = launch_fused<1, CAP, MODE, 1, 64>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break
      case 12108: SQ_LAUNCH_H(8, sq::MODE_MX);
      case 12120: SQ_LAUNCH_H(20, sq::MODE_MX);
      case 12132: SQ_LAUNCH_H(32, sq::MODE_MX);
      case 11108: SQ_LAUNCH_H(8, sq::MODE_F8);
      case 11120: SQ_LAUNCH_H(20, sq::MODE_F8);
      case 11132: SQ_LAUNCH_H(32, sq::MODE_F8);
      case 10108: SQ_LAUNCH_H(8, sq::MODE_BF16);
      case 10120: SQ_LAUNCH_H(20, sq::MODE_BF16);
      case 10132: SQ_LAUNCH_H(32, sq::MODE_BF16);
#undef SQ_LAUNCH_H
      case 2108: SQ_LAUNCH(1, 8, sq::MODE_MX);
      case 2120: SQ_LAUNCH(1, 20, sq::MODE_MX);
      case 2132: SQ_LAUNCH(1, 32, sq::MODE_MX);
      case 2208: SQ_LAUNCH(2, 8, sq::MODE_MX);
      case 2220: SQ_LAUNCH(2, 20, sq::MODE_MX);
      case 2232: SQ_LAUNCH(2, 32, sq::MODE_MX);
      case 1108: SQ_LAUNCH(1, 8, sq::MODE_F8);
      case 1120: SQ_LAUNCH(1, 20, sq::MODE_F8);
      case 1132: SQ_LAUNCH(1, 32, sq::MODE_F8);
      case 1208: SQ_LAUNCH(2, 8, sq::MODE_F8);
      case 1220: SQ_LAUNCH(2, 20, sq::MODE_F8);
      case 1232: SQ_LAUNCH(2, 32, sq::MODE_F8);
      case 108: SQ_LAUNCH(1, 8, sq::MODE_BF16);
      case 120: SQ_LAUNCH(1, 20, sq::MODE_BF16);
      case 132: SQ_LAUNCH(1, 32, sq::MODE_BF16);
      case 1408: e = launch_fused<2, 8, sq::MODE_F8, 4>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break;
      case 1420: e = launch_fused<2, 20, sq::MODE_F8, 4>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break;
      case 1432: e = launch_fused<2, 32, sq::MODE_F8, 4>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break;
      case 408: e = launch_fused<2, 8, sq::MODE_BF16, 4>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break;
      case 420: e = launch_fused<2, 20, sq::MODE_BF16, 4>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break;
      case 432: e = launch_fused<2, 32, sq::MODE_BF16, 4>(pl, ctx->num_sms, th, tw, tsa, tsb, fp, st); break;
      case 208: SQ_LAUNCH(2, 8, sq::MODE_BF16);
      case 220: SQ_LAUNCH(2, 20, sq::MODE_BF16);
      default: SQ_LAUNCH(2, 32, sq::MODE_BF16);
    }
#undef SQ_LAUNCH
    if (e != cudaSuccess) return set_err(ctx, SQ_ERR_CUDA, "fused kernel launch failed: %s", cudaGetErrorString(e));
    if (pev) cudaEventRecord(pev[1], st);

    sq::FinalizeParams fin = {};
    fin.T = T; fin.V = V; fin.k = k; fin.cap = pl.topk_cap; fin.num_chunks = pl.num_chunks;
    fin.targets = targets;
    fin.part_m = ctx->part_m; fin.part_s = ctx->part_s; fin.part_u = ctx->part_u;
    fin.part_cs = ctx->part_cs; fin.part_cu = ctx->part_cu;
    fin.part_topv = ctx->part_topv; fin.part_topi = ctx->part_topi; fin.zt = ctx->zt;
    fin.lse = lse; fin.target_logprob = lp; fin.entropy = ent; fin.conf = conf;
    fin.topk_logprob = o->topk_logprob; fin.topk_index = o->topk_index;
    fin.chunks_per_rank = pl.num_chunks; fin.num_ranks = 1;   // (rank_off[0] = 0)
    fin.vocab_offset = vocab_offset;
    // a small run (decode-shaped): kernel 2 would be pure launch latency, the finalize kernel's last CTA does its work
    const bool tail = !shard_state && B > 0 && T <= sq::FIN_TAIL_MAX_T;
    if (tail) {
      fin.tail_B = B; fin.tail_window = window; fin.tail_cu = cu_seqlens; fin.tail_counter = ctx->tail_counter;
      fin.tail_out_lp = o->seq_mean_logprob; fin.tail_out_ent = o->seq_mean_entropy; fin.tail_out_conf = o->seq_mean_conf;
      fin.tail_out_min = o->seq_min_window_conf;
    }
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
      else SQ_CUDA(ctx, launch_wide_finalize<true>(pl.topk_cap, T, st, fin));
    } else if (pl.num_chunks <= 32) {
      SQ_CUDA(ctx, launch_pdl(sq::sq_finalize_kernel<1, false>, fgrid, fblock, 0, st, fin));
    } else {
      SQ_CUDA(ctx, launch_wide_finalize<false>(pl.topk_cap, T, st, fin));
    }
    ctx->launches += 2;
    SQ_CUDA(ctx, cudaGetLastError());
    if (pev) cudaEventRecord(pev[2], st);
    if (pev && (B == 0 || tail)) { cudaEventRecord(pev[3], st); ++ctx->ev_count; }   // no kernel 2 follows (shard runs, B = 0, small runs)
    if (tail) { ctx->reduce_form = SQ_REDUCE_FORM_TAIL; return SQ_OK; }
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
    if (ctx->profiling && T > 0) { cudaEventRecord(ctx->ev[ctx->ev_count % SQ_PROFILE_RING][3], st); ++ctx->ev_count; }
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

// ------------------------------------------------------------------------------------------ block-scaled (MX) variant
static void mx_geometry(int64_t rows, int d, int operand, int* blk_rows, int* pieces, int64_t* num_blk, int64_t* kblocks) {
  *blk_rows = operand == SQ_MX_OPERAND_W ? sq::BLOCK_N_MX : sq::BLOCK_M;
  *pieces = (*blk_rows + 127) / 128;
  *num_blk = cdiv64(rows, *blk_rows);
  *kblocks = cdiv64(d, sq::BLOCK_K_F8);
}

extern "C" int64_t sq_score_mx_scale_bytes(int64_t num_rows, int d, int operand) {
  if (num_rows < 0 || d < 1 || (operand != SQ_MX_OPERAND_H && operand != SQ_MX_OPERAND_W)) return -1;
  int blk_rows, pieces; int64_t num_blk, kblocks;
  mx_geometry(num_rows, d, operand, &blk_rows, &pieces, &num_blk, &kblocks);
  return kblocks * num_blk * pieces * 512;
}

extern "C" int sq_score_quantize_mx(sq_score_ctx* ctx, const void* X, int64_t num_rows, int operand, void* q_out, void* sf_out,
                                    void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_rows < 0 || (operand != SQ_MX_OPERAND_H && operand != SQ_MX_OPERAND_W)) return set_err(ctx, SQ_ERR_INVALID_ARG, "bad row count or operand");
  if (num_rows == 0) return SQ_OK;
  if (!X || !q_out || !sf_out) return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument");
  if (ctx->cfg.d % 16 != 0) return set_err(ctx, SQ_ERR_UNSUPPORTED, "the MX variant needs d %% 16 == 0 (TMA 16-byte row strides)");
  if (((uintptr_t)X & 15) || ((uintptr_t)q_out & 15) || ((uintptr_t)sf_out & 15))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "X, q_out and sf_out must be 16-byte aligned");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  sq::QuantMxParams qp = {};
  int64_t kblocks;
  mx_geometry(num_rows, ctx->cfg.d, operand, &qp.blk_rows, &qp.pieces, &qp.num_blk, &kblocks);
  qp.X = static_cast<const uint4*>(X); qp.Q = static_cast<uint2*>(q_out); qp.SF = static_cast<uint8_t*>(sf_out);
  qp.rows = num_rows; qp.d = ctx->cfg.d;
  // slots no row or k-block reaches (ragged last blocks) scale zero-filled codes: any value but NaN (0xFF) would do
  SQ_CUDA(ctx, cudaMemsetAsync(sf_out, 0, (size_t)(kblocks * qp.num_blk * qp.pieces * 512), st));
  const unsigned ctas = (unsigned)std::min<int64_t>(cdiv64(num_rows, 8), (int64_t)ctx->num_sms * 8);
  sq::sq_quant_mx_kernel<<<ctas, 256, 0, st>>>(qp);
  ctx->launches += 1;
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
}

extern "C" int sq_score_run_mx(sq_score_ctx* ctx, const void* Hq, const void* h_sf, const void* Wq, const void* w_sf,
                               const int32_t* targets, const int32_t* cu_seqlens, int num_tokens, int num_seqs, int k,
                               int window, const sq_score_outputs* outputs, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_tokens > 0 && (!h_sf || !w_sf)) return set_err(ctx, SQ_ERR_INVALID_ARG, "h_sf and w_sf are required");
  if (num_tokens > 0 && (((uintptr_t)h_sf & 15) || ((uintptr_t)w_sf & 15))) return set_err(ctx, SQ_ERR_INVALID_ARG, "h_sf and w_sf must be 16-byte aligned");
  return run_impl(ctx, Hq, Wq, targets, cu_seqlens, num_tokens, num_seqs, k, window, outputs, stream, nullptr, 0, 0, nullptr,
                  nullptr, nullptr, 0, h_sf, w_sf);
}

// ------------------------------------------------------------------------------------------ vocab-parallel (8(f)-4)
extern "C" int64_t sq_score_shard_state_bytes(int64_t num_tokens, int k) {
  if (num_tokens < 0 || k < 1 || k > SQ_MAX_K) return -1;
  return shard_state_words(num_tokens, topk_cap_for(k)) * 4;
}

extern "C" int sq_score_run_shard(sq_score_ctx* ctx, const void* H, const void* W_shard, int shard_rows, int vocab_offset,
                                  const int32_t* targets, int num_tokens, int k, void* state_out, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (vocab_offset < 0) return set_err(ctx, SQ_ERR_INVALID_ARG, "vocab_offset must be >= 0");
  if (shard_rows < 1 || shard_rows > ctx->cfg.vocab)
    return set_err(ctx, SQ_ERR_INVALID_ARG, "shard_rows = %d outside 1..cfg.vocab = %d", shard_rows, ctx->cfg.vocab);
  if (k > shard_rows) return set_err(ctx, SQ_ERR_INVALID_ARG, "k = %d exceeds the shard's %d rows", k, shard_rows);
  if (num_tokens > 0 && !state_out) return set_err(ctx, SQ_ERR_INVALID_ARG, "state_out is null");
  if (num_tokens == 0) return SQ_OK;
  return run_impl(ctx, H, W_shard, targets, nullptr, num_tokens, 0, k, 1, nullptr, stream, nullptr, 0, vocab_offset,
                  static_cast<float*>(state_out), nullptr, nullptr, shard_rows);
}

extern "C" int sq_score_neutral_shard_state(sq_score_ctx* ctx, int num_tokens, int k, void* state_out, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_tokens < 0 || k < 1 || k > SQ_MAX_K) return set_err(ctx, SQ_ERR_INVALID_ARG, "T >= 0 and 1 <= k <= %d required", SQ_MAX_K);
  if (num_tokens == 0) return SQ_OK;
  if (!state_out) return set_err(ctx, SQ_ERR_INVALID_ARG, "state_out is null");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  const int cap = topk_cap_for(k);
  const int64_t words = shard_state_words(num_tokens, cap);
  const unsigned grid = (unsigned)std::min<int64_t>(cdiv64(words, 256), (int64_t)ctx->num_sms * 8);
  sq::sq_neutral_state_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<float*>(state_out), num_tokens, cap);
  ctx->launches += 1;
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
}

// `states`: the R packed states back to back, or null with `peers`: R pointers to one packed state each (HOST array)
static int merge_impl(sq_score_ctx* ctx, const void* states, const void* const* peers, int num_shards, const int32_t* vocab_starts,
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
  if (T > 0 && ((!states && !peers) || !targets)) return set_err(ctx, SQ_ERR_INVALID_ARG, "states and targets are required");
  if (T > 0 && peers)
    for (int r = 0; r < num_shards; ++r)
      if (!peers[r] || ((uintptr_t)peers[r] & 3)) return set_err(ctx, SQ_ERR_INVALID_ARG, "state pointer %d is null or not 4-byte aligned", r);
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
    fin.chunks_per_rank = 1; fin.num_ranks = num_shards;
    const void* base = peers ? peers[0] : states;
    for (int r = 0; r < num_shards; ++r)   // distance of rank r's state from rank 0's, in words (any sign)
      fin.rank_off[r] = peers ? (long long)((intptr_t)peers[r] - (intptr_t)base) / 4 : (long long)r * shard_state_words(T, cap);
    for (int r = 0; r <= num_shards; ++r) fin.vstart[r] = vocab_starts[r];
    fin.targets = targets;
    set_state_pointers(fin, const_cast<float*>(static_cast<const float*>(base)), T, cap, /*as_output=*/false);
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

extern "C" int sq_score_merge_shards(sq_score_ctx* ctx, const void* states, int num_shards, const int32_t* vocab_starts,
                                     const int32_t* targets, const int32_t* cu_seqlens, int num_tokens, int num_seqs,
                                     int k, int window, const sq_score_outputs* o, void* stream) {
  return merge_impl(ctx, states, nullptr, num_shards, vocab_starts, targets, cu_seqlens, num_tokens, num_seqs, k, window, o, stream);
}

extern "C" int sq_score_merge_shards_peer(sq_score_ctx* ctx, const void* const* state_ptrs, int num_shards,
                                          const int32_t* vocab_starts, const int32_t* targets, const int32_t* cu_seqlens,
                                          int num_tokens, int num_seqs, int k, int window, const sq_score_outputs* o, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (!state_ptrs) return set_err(ctx, SQ_ERR_INVALID_ARG, "state_ptrs is null");
  return merge_impl(ctx, nullptr, state_ptrs, num_shards, vocab_starts, targets, cu_seqlens, num_tokens, num_seqs, k, window, o, stream);
}

extern "C" int sq_score_debug_fill_workspace(sq_score_ctx* ctx, int value, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const sq_score_config& c = ctx->cfg;
  const bool ro = (c.flags & SQ_FLAG_REDUCE_ONLY) != 0;
  const int64_t rows = ro ? 1 : ws_rows_for(c), T = c.max_tokens;
  struct Buf { void* p; int64_t bytes; };
  const Buf bufs[] = {
      {ctx->part_m, rows * 4}, {ctx->part_s, rows * 4}, {ctx->part_u, rows * 4}, {ctx->part_cs, rows * 4}, {ctx->part_cu, rows * 4},
      {ctx->part_topv, rows * ctx->cap_max * 4}, {ctx->part_topi, rows * ctx->cap_max * 4}, {ctx->zt, (ro ? 1 : T) * 4},
      {ctx->gang_ctr, 256 * 4}, {ctx->thr_pub, (ro ? 1 : (int64_t)THR_MAX_CHUNKS * T) * 4},
      {ctx->tok_lse, (ro ? 1 : T) * 4}, {ctx->tok_lp, (ro ? 1 : T) * 4}, {ctx->tok_ent, (ro ? 1 : T) * 4}, {ctx->tok_conf, (ro ? 1 : T) * 4},
      {ctx->tile_base, ((int64_t)c.max_seqs + 1) * 4}, {ctx->amax_bits, 4}, {ctx->red_sum, ctx->red_tiles_max * 16},
      {ctx->tile_seq, ctx->red_tiles_max * 4}, {ctx->red_min, ctx->red_tiles_max * 4}, {ctx->seq_stage, 4 * (int64_t)c.max_seqs * 4},
      {ctx->pos_base, ((int64_t)c.max_seqs + 1) * 4},
      {ctx->h_stage, ctx->h_stage ? T * (int64_t)c.d * 2 : 0}, {ctx->tgt_stage, ctx->tgt_stage ? T * 4 : 0},
      {ctx->cu_stage, ctx->cu_stage ? ((int64_t)c.max_seqs + 1) * 4 : 0}, {ctx->h_flags, ctx->h_flags ? HOST_FLAGS_PER_RUN * 4 : 0}};
  for (const Buf& b : bufs)
    if (b.p && b.bytes > 0) SQ_CUDA(ctx, cudaMemsetAsync(b.p, value, (size_t)b.bytes, st));
  SQ_CUDA(ctx, cudaMemsetAsync(ctx->seq_done, 0, (size_t)c.max_seqs * sizeof(int), st));   // invariant: zero between runs
  return SQ_OK;
}

extern "C" int sq_score_set_profiling(sq_score_ctx* ctx, int enable) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  if (enable && !ctx->ev) {
    ctx->ev = new (std::nothrow) cudaEvent_t[SQ_PROFILE_RING][4]();
    if (!ctx->ev) return set_err(ctx, SQ_ERR_NOMEM, "host allocation failed");
    for (int i = 0; i < SQ_PROFILE_RING; ++i)
      for (auto& e : ctx->ev[i]) SQ_CUDA(ctx, cudaEventCreate(&e));
  }
  ctx->profiling = enable ? 1 : 0;
  ctx->ev_count = ctx->ev_read = 0;
  return SQ_OK;
}

static int read_run_times(sq_score_ctx* ctx, int64_t run, float* ms3) {
  cudaEvent_t* e = ctx->ev[run % SQ_PROFILE_RING];
  SQ_CUDA(ctx, cudaEventSynchronize(e[3]));
  for (int i = 0; i < 3; ++i) SQ_CUDA(ctx, cudaEventElapsedTime(&ms3[i], e[i], e[i + 1]));
  return SQ_OK;
}

extern "C" int sq_score_kernel_times(sq_score_ctx* ctx, float* ms3) {
  if (!ctx || !ms3) return SQ_ERR_INVALID_ARG;
  if (!ctx->profiling || ctx->ev_count == 0) return set_err(ctx, SQ_ERR_INVALID_ARG, "no profiled run recorded");
  return read_run_times(ctx, ctx->ev_count - 1, ms3);
}

extern "C" int sq_score_profile_read(sq_score_ctx* ctx, float* ms, int capacity, int* num_runs) {
  if (!ctx || !ms || !num_runs || capacity < 0) return SQ_ERR_INVALID_ARG;
  *num_runs = 0;
  if (!ctx->profiling) return set_err(ctx, SQ_ERR_INVALID_ARG, "profiling is off");
  int64_t first = std::max(ctx->ev_read, ctx->ev_count - SQ_PROFILE_RING);
  first = std::max(first, ctx->ev_count - capacity);
  for (int64_t r = first; r < ctx->ev_count; ++r) {
    const int rc = read_run_times(ctx, r, ms + 3 * (r - first));
    if (rc != SQ_OK) return rc;
  }
  *num_runs = (int)(ctx->ev_count - first);
  ctx->ev_read = ctx->ev_count;
  return SQ_OK;
}

static int need_staging(sq_score_ctx* ctx) {
  if (ctx->h_stage && ctx->copy_stream) return SQ_OK;
  return set_err(ctx, SQ_ERR_INVALID_ARG, "this call needs a ctx created with SQ_FLAG_STAGING (no run allocates)");
}

// ------------------------------------------------------------------------------------------ positions (8(f)-2)
extern "C" int sq_score_positions_host(const int32_t* query_lens, const int32_t* traj_lens, int num_seqs, int32_t* pos_out,
                                       int64_t pos_capacity, int32_t* cu_out, int64_t* num_tokens_out) {
  if (num_seqs < 0 || pos_capacity < 0 || !cu_out || (num_seqs > 0 && (!query_lens || !traj_lens))) return SQ_ERR_INVALID_ARG;
  int64_t t = 0, base = 0;
  cu_out[0] = 0;
  for (int b = 0; b < num_seqs; ++b) {
    const int64_t q = query_lens[b], n = traj_lens[b];
    if (q < 0 || n < 0 || (n > 0 && q < 1)) return SQ_ERR_INVALID_ARG;   // no state predicts the trajectory's first token
    if (t + n > pos_capacity || base + q + n > INT32_MAX || (n > 0 && !pos_out)) return SQ_ERR_INVALID_ARG;
    for (int64_t i = 0; i < n; ++i) pos_out[t + i] = (int32_t)(base + q - 1 + i);
    t += n;
    base += q + n;
    cu_out[b + 1] = (int32_t)t;
  }
  if (num_tokens_out) *num_tokens_out = t;
  return SQ_OK;
}

extern "C" int sq_score_positions(sq_score_ctx* ctx, const int32_t* query_lens, const int32_t* traj_lens, int num_seqs,
                                  int num_tokens, int32_t* pos_out, int32_t* cu_out, int32_t* status_out, void* stream) {
  if (!ctx) return SQ_ERR_INVALID_ARG;
  if (num_seqs < 0 || num_tokens < 0 || num_seqs > ctx->cfg.max_seqs || num_tokens > ctx->cfg.max_tokens)
    return set_err(ctx, SQ_ERR_INVALID_ARG, "B / T out of range for this ctx");
  if (!cu_out || (num_seqs > 0 && (!query_lens || !traj_lens)) || (num_tokens > 0 && !pos_out))
    return set_err(ctx, SQ_ERR_INVALID_ARG, "null pointer argument");
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  sq::PositionsParams pp = {};
  pp.query_lens = query_lens; pp.traj_lens = traj_lens; pp.B = num_seqs; pp.num_tokens = num_tokens;
  pp.pos = pos_out; pp.cu = cu_out; pp.base = ctx->pos_base; pp.status = status_out;
  sq::sq_positions_scan_kernel<<<1, 1024, 0, st>>>(pp);
  ctx->launches += 1;
  if (num_seqs > 0 && num_tokens > 0) {
    sq::sq_positions_fill_kernel<<<(unsigned)num_seqs, 256, 0, st>>>(pp);
    ctx->launches += 1;
  }
  SQ_CUDA(ctx, cudaGetLastError());
  return SQ_OK;
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
  int rc = need_staging(ctx);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  rc = sq_score_prepare(ctx, X, num_rows, pos, num_tokens, gain, eps, ctx->h_stage, stream);
  if (rc != SQ_OK) return rc;
  return run_impl(ctx, ctx->h_stage, W, targets, cu_seqlens, num_tokens, num_seqs, k, window, outputs, stream, nullptr, 0);
}

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
  if (need_staging(ctx) != SQ_OK) return SQ_ERR_INVALID_ARG;
  SQ_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
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
