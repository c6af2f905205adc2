/*
 * sq_score.h -- C ABI of the B200-native fused LM-head scoring library (libsq_score.so).
 *
 * The hot path is the prefill-side token-scoring pass behind SQUEEZE EVOLVE's confidence-based
 * routing (arxiv 2604.07725):
 *   - per-token top-K_l confidence  c(i) = -(1/K_l) * sum_{j<=K_l} log p(v_j^(i) | t_<i, Q)     Eq. 3
 *   - per-trajectory confidence     C(tau) = (1/|tau|) * sum_i c(i)                             Eq. 4
 *   - "cross-model log-probabilities" of the trajectory tokens
 *   - one prefill-only pass over the N batched candidates, reduced on the GPU so that only
 *     scalars per trajectory leave the device
 *   - entropy and the sliding-window minimum are defined by BASELINE.json `north_star`.
 *
 * Given final hidden states H[T,d] and an LM head W[V,d] (bf16, row-major = K-major) the library
 * never materialises the [T,V] logits: kernel 1 fuses the vocabulary GEMM (tcgen05 / TMEM / TMA,
 * sm_100a) with an online logsumexp, target-logit capture, entropy and streaming top-k; a merge
 * kernel combines vocab-chunk partial states; kernel 2 does the per-sequence varlen reductions.
 *
 * Conventions
 *   - every function returns 0 (SQ_OK) or a negative SQ_ERR_* code; nothing aborts or throws.
 *   - every `sq_score_run*` call, `sq_score_reduce`, `sq_score_prepare`, ... is ASYNCHRONOUS on `stream`
 *     (a cudaStream_t passed as void*) and does no host synchronisation and NO ALLOCATION of any kind:
 *     all workspace, staging buffers, streams and events are owned by the ctx and created by
 *     `sq_score_create` from max_tokens / max_seqs / max_k / flags.  (Only `sq_score_set_profiling`
 *     creates events, outside any run.)
 *   - kernel 1 is a persistent kernel whose clusters wait for one another (gang barriers): all of them
 *     must be resident at once.  `sq_score_create` asks the occupancy calculator how many clusters the
 *     device can hold and plans for that many; the device must not be running other kernels that
 *     occupy SMs while a run executes.  A wait that lasts longer than cfg.wait_seconds traps (the run
 *     fails with a sticky CUDA error) instead of hanging the device.
 *   - pointers marked DEVICE must be device memory on ctx's device; HOST pointers are host memory
 *     (pinned for true async copies).  The library never frees or keeps caller buffers beyond the
 *     work it enqueued.
 *   - H and W: bf16, contiguous, 16-byte aligned, d % 8 == 0 (TMA 16-byte stride rule).
 *   - cu_seqlens[0] = 0, non-decreasing, cu_seqlens[B] = T.  Device-side contents are trusted.
 *   - targets[t] outside [0, V) means "no target": target_logprob[t] = 0 and the token is left out
 *     of seq_mean_logprob (numerator and denominator).
 *   - empty sequences give NaN aggregates; window' = min(window, L), stride 1, full windows only.
 *   - one ctx per host thread / stream.  There is no CPU fallback: without a B200-class device
 *     `sq_score_create` fails with SQ_ERR_CUDA / SQ_ERR_UNSUPPORTED.
 */
#ifndef SQ_SCORE_H_
#define SQ_SCORE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SQ_OK                 0
#define SQ_ERR_INVALID_ARG   -1   /* null pointer, size out of range, k > max_k, ...              */
#define SQ_ERR_UNSUPPORTED   -2   /* shape or device the kernels do not cover (d % 8, not sm_100) */
#define SQ_ERR_CUDA          -3   /* a CUDA runtime/driver call failed; see sq_score_last_error   */
#define SQ_ERR_NOMEM         -4   /* workspace allocation failed                                  */

#define SQ_MAX_K             32   /* largest K_l the streaming top-k supports                     */

#define SQ_FLAG_REDUCE_ONLY   1   /* ctx serves sq_score_reduce only: no kernel-1 workspace is
                                     allocated and sq_score_run / run_host return INVALID_ARG    */
#define SQ_FLAG_STAGING       2   /* also allocate, at create, what sq_score_run_host and
                                     sq_score_run_x need: an H buffer [max_tokens, d] bf16, staged
                                     targets / cu_seqlens, arrival flags, a copy stream and its
                                     events.  Without it those two calls return INVALID_ARG.     */

#define SQ_DEBUG_PREPARE_TWO_PASS   8   /* sq_score_prepare: two-pass kernel instead of register-resident rows */
#define SQ_DEBUG_NO_SHARED_BOUND   16   /* kernel 1: no shared top-k bound between the chunks of a row     */
#define SQ_DEBUG_REDUCE_TILES      32   /* kernel 2: three-launch tile form                                */
#define SQ_DEBUG_REDUCE_FUSED      64   /* kernel 2: single-launch form                                    */
#define SQ_DEBUG_FINALIZE_WARP    128   /* finalize: one warp per row                                      */
#define SQ_DEBUG_REDUCE_STREAM    256   /* kernel 2: streaming form wherever it applies                    */
#define SQ_DEBUG_ALL (8 | 16 | 32 | 64 | 128 | 256)

#define SQ_MAX_CHUNKS       160   /* vocab chunks per row at most                                 */
#define SQ_MAX_VOCAB   14679840   /* largest V: 65535 vocab tiles (16-bit tile indices) of the narrowest
                                     tile, the MX variant's 224 columns                           */

typedef struct sq_score_ctx sq_score_ctx;   /* opaque */

/* Fixed per context (one scorer model = one LM head shape). */
typedef struct {
  int     device;       /* CUDA device ordinal                                                    */
  int     d;            /* hidden size, d % 8 == 0                                                */
  int     vocab;        /* V                                                                      */
  int64_t max_tokens;   /* largest T of any run (sizes the partial-state workspace)               */
  int     max_seqs;     /* largest B of any run                                                   */
  int     max_k;        /* largest k of any run, 1..SQ_MAX_K                                      */
  int     cta_group;    /* 0 = default (CTA pairs, UMMA M=256; single CTA when T <= 128);
                           1 = always single-CTA UMMA (M=128); 2 = always CTA pairs               */
  int     num_chunks;   /* 0 = planner's choice; >0 forces the number of vocab chunks per row     */
  int     group_m;      /* 0 = planner's choice (10..14, 12 preferred): gang size = clusters that
                           share one W stream; >0 forces it                                       */
  int     flags;        /* SQ_FLAG_*                                                              */
  int     wait_seconds; /* how long a device-side wait (pipeline barrier, gang barrier, H arrival
                           flag) may last before kernel 1 traps: 0 = default (60 s), < 0 = for ever.
                           One limit for every wait: in sq_score_run_host the copy of the whole H must
                           land within it                                                          */
  /* The three below select between code paths that give the SAME results; 0 = the library's choice.  Tests force
     every path through them; a user has no reason to set them. */
  int     debug_flags;  /* SQ_DEBUG_* bits                                                        */
  int     cluster4;     /* quad scheduling with W multicast in kernel 1: 0 = runs of more than 200 000
                           tokens (default), 1 = every run of more than 4096 tokens, -1 = never       */
  int     region_mult;  /* length of kernel 1's regions (token tiles between barriers across all gangs) in
                           units of the gang sizes' common multiple: 0 = default (~160 tiles), > 0 forced,
                           -1 = no region barrier                                                  */
} sq_score_config;

/* Output pointers of one run.  Per-token pointers may be NULL (= not wanted; the ctx keeps the
 * 12 B/token kernel 2 needs in its own scratch).  Per-sequence pointers are required. */
typedef struct {
  float   *lse;                 /* DEVICE [T]   logsumexp_v z[t,v]                                */
  float   *target_logprob;      /* DEVICE [T]   z[t,targets[t]] - lse[t]     */
  float   *entropy;             /* DEVICE [T]   -sum_v p log p, nats                              */
  float   *conf;                /* DEVICE [T]   c(i), Eq. 3    */
  float   *topk_logprob;        /* DEVICE [T,k] row-major, descending                             */
  int32_t *topk_index;          /* DEVICE [T,k] vocabulary ids of topk_logprob                    */
  float   *seq_mean_logprob;    /* DEVICE [B]   mean target_logprob over valid targets            */
  float   *seq_mean_entropy;    /* DEVICE [B]                                                     */
  float   *seq_mean_conf;       /* DEVICE [B]   C(tau), Eq. 4    */
  float   *seq_min_window_conf; /* DEVICE [B]   min over windows of the window-mean of c(i)       */
} sq_score_outputs;

/* How a run of T tokens is cut into work units (host logic, no GPU needed).
 * The clusters are split into num_gangs gangs: gangs [0, gangs_big) have gang_size + 1 members, the rest
 * gang_size.  Gang i owns vocab chunks [i * chunks_per_gang, (i+1) * chunks_per_gang) and walks the token
 * tiles in batches of its own size; chunk c sweeps vocab tiles [chunk_vtile[c], chunk_vtile[c+1]).        */
typedef struct {
  int cta_group;        /* 1 or 2                                                                 */
  int rows_per_tile;    /* 128 * cta_group token rows per work unit                               */
  int m_tiles;          /* ceil(T / rows_per_tile)                                                */
  int num_vtiles;       /* ceil(V / 256)                                                          */
  int num_k_blocks;     /* ceil(d / 64)                                                           */
  int num_chunks;       /* vocab chunks per row = num_gangs * chunks_per_gang (partial states merged
                           by the finalize kernel)                                                */
  int chunks_per_gang;  /* chunks a gang's vocabulary stripe is cut into (1 unless num_chunks is forced) */
  int tiles_per_chunk;  /* width of the widest chunk, in vocab tiles                               */
  int num_units;        /* m_tiles * num_chunks                                                   */
  int num_clusters;     /* clusters the device can hold (SMs / cta_group, or what create() found)  */
  int num_gangs;
  int gang_size;        /* members of the smaller gangs                                           */
  int gangs_big;        /* gangs with gang_size + 1 members                                       */
  int clusters_used;    /* num_gangs * gang_size + gangs_big = clusters launched                  */
  int max_batches;      /* batches of token tiles the smallest gang walks: ceil(m_tiles / gang_size) */
  int topk_cap;         /* compiled top-k list capacity used for this k (8, 20 or 32)             */
  int chunk_vtile[SQ_MAX_CHUNKS + 1];
} sq_score_plan_t;

/* Creates a context on cfg->device and allocates its workspace (and, with SQ_FLAG_STAGING, the staging of
 * sq_score_run_host / sq_score_run_x); queries how many clusters of kernel 1 the device can hold at once.
 * Errors: INVALID_ARG (null, sizes <= 0, max_k out of range), UNSUPPORTED (d % 8 != 0, vocab > SQ_MAX_VOCAB, device
 * is not compute capability 10.x, or it cannot hold even one cluster of kernel 1), CUDA, NOMEM.  On error
 * *out is NULL. */
int sq_score_create(const sq_score_config *cfg, sq_score_ctx **out);

/* Scores T tokens: enqueues kernel 1 (fused GEMM + statistics), the merge/finalize kernel and kernel 2 on
 * `stream` (runs of at most 256 tokens -- decode-shaped -- do kernel 2's work in the finalize kernel's last CTA:
 * two launches instead of three).
 *   H          DEVICE bf16 [T,d]       final hidden states; row t predicts targets[t] (the caller
 *                                      does the next-token shift and packs only trajectory tokens)
 *   W          DEVICE bf16 [V,d]       LM head
 *   targets    DEVICE int32 [T]
 *   cu_seqlens DEVICE int32 [B+1]
 *   k          1..min(max_k, V)        K_l of Eq. 3
 *   window     >= 1
 * T == 0 or B == 0 is legal (nothing / NaNs are written).
 * Errors: INVALID_ARG (null required pointer, T > max_tokens, B > max_seqs, k or window out of
 * range, misaligned H/W), CUDA. */
int sq_score_run(sq_score_ctx *ctx, const void *H, const void *W, const int32_t *targets,
                 const int32_t *cu_seqlens, int num_tokens, int num_seqs, int k, int window,
                 const sq_score_outputs *outputs, void *stream);

/* End-to-end form with HOST inputs and HOST results: copies targets and cu_seqlens to ctx-owned
 * device staging buffers, streams H in on a ctx-owned copy stream in blocks of rows (ascending, each
 * block followed by an arrival flag) WHILE kernel 1 runs -- its producers wait for the flag of the
 * rows they are about to load, so the transfer hides behind the GEMM -- runs the same kernels, and
 * copies the 4*B per-sequence scalars back (order: mean_logprob[B], mean_entropy[B], mean_conf[B],
 * min_window_conf[B]).  W stays on the device (it is the resident model weight).  Asynchronous on
 * `stream` (which also waits for the copy stream); the caller synchronises `stream` before reading
 * seq_out_host or reusing the host buffers.  Pinned host memory is needed for the overlap; pageable
 * memory works but its copies are staged by the runtime.  Needs a ctx created with SQ_FLAG_STAGING.
 * Errors: as sq_score_run; INVALID_ARG without SQ_FLAG_STAGING. */
int sq_score_run_host(sq_score_ctx *ctx, const void *H_host, const void *W_dev,
                      const int32_t *targets_host, const int32_t *cu_seqlens_host,
                      int num_tokens, int num_seqs, int k, int window,
                      float *seq_out_host, void *stream);

/* Kernel 2 alone: per-sequence varlen reductions of caller-provided per-token arrays.
 *   target_logprob, entropy, conf  DEVICE float [T]
 *   targets                        DEVICE int32 [T] or NULL (NULL = every target valid)
 *   seq_* outputs                  DEVICE float [B]
 * Errors: INVALID_ARG, CUDA. */
int sq_score_reduce(sq_score_ctx *ctx, const float *target_logprob, const float *entropy,
                    const float *conf, const int32_t *targets, const int32_t *cu_seqlens,
                    int64_t num_tokens, int num_seqs, int window,
                    float *seq_mean_logprob, float *seq_mean_entropy, float *seq_mean_conf,
                    float *seq_min_window_conf, void *stream);

/* Kernel 2 for callers that cannot allocate device memory -- and therefore cannot call sq_score_create, which
 * cudaMallocs the workspace.  Two kinds of caller are meant:
 *   - a plug-in inside a serving engine that has already handed (nearly) all free HBM to its own pool (KV cache,
 *     activation arena): a cudaMalloc from a library fails there, or eats into a budget the engine believes it owns;
 *   - code on a latency-critical path (a decode loop, a scheduler callback): cudaMalloc and cudaFree may synchronise
 *     the whole device, so one allocation stalls every stream of the process.
 * This call needs NO ctx and calls no cudaMalloc, cudaFree or allocating library routine, neither on its first call nor
 * later.  It computes what sq_score_reduce computes (same kernel body, the single-launch form; the same bits), with the
 * tile partials and per-sequence counters the kernel needs kept in a fixed array inside the library's device image
 * instead of a ctx workspace.  That array costs about 186 KB of HBM on every GPU that loads libsq_score.so, from load to
 * process exit, whether or not this call is ever made; in exchange the sizes are capped:
 *     num_tokens <= SQ_STATIC_MAX_TOKENS,   num_seqs <= SQ_STATIC_MAX_SEQS
 * and anything larger is refused with SQ_ERR_INVALID_ARG (message via sq_score_last_error(NULL)); nothing is launched.
 *
 * It runs on the calling thread's CURRENT device (cudaSetDevice is the caller's business; all pointers DEVICE memory of
 * that device), asynchronously on `stream`: one 4*num_seqs-byte cudaMemsetAsync (the counters must start at zero, and a
 * call that died half way may have left some behind) and one kernel launch.
 *   target_logprob, entropy, conf  DEVICE float [num_tokens]
 *   targets      DEVICE int32 [num_tokens] or NULL (NULL = every target valid)
 *   cu_seqlens   DEVICE int32 [num_seqs+1]
 *   vocab        targets outside [0, vocab) are "no target" (sq_score_reduce takes this from its ctx); ignored when
 *                targets == NULL
 *   seq_*        DEVICE float [num_seqs], written by this call; the caller owns every buffer it passes
 * First call on each device: looks up the device address of the array and the SM count and raises the kernel's
 * dynamic-shared-memory limit (host-side driver calls, no allocation).  Make that first call early, at start-up and
 * before any stream capture begins; later calls only enqueue work.
 * One array per device, shared by every call in the process and keeping what the last call left: two calls whose
 * kernels may overlap on the GPU (different streams with no ordering between them, several host threads) RACE on it
 * and give wrong results.  Put every call on one stream, or order the streams with events.
 * Errors: INVALID_ARG (null pointer, negative size, window < 1, vocab < 1 with targets, a size beyond the maximum),
 * CUDA (no device, not an sm_100 device, a runtime call failed).  Messages: sq_score_last_error(NULL), per thread. */
#define SQ_STATIC_MAX_TOKENS 4194304   /* 2^22 tokens per call                                    */
#define SQ_STATIC_MAX_SEQS      4096   /* sequences per call                                      */
int sq_score_reduce_static(const float *target_logprob, const float *entropy, const float *conf,
                           const int32_t *targets, const int32_t *cu_seqlens, int64_t num_tokens, int num_seqs,
                           int vocab, int window, float *seq_mean_logprob, float *seq_mean_entropy,
                           float *seq_mean_conf, float *seq_min_window_conf, void *stream);

/* The step before the path: gathers the hidden states that predict the scored
 * tokens and applies the scorer's final RMSNorm,
 *     H_out[t,:] = bf16( x / sqrt(mean_j x_j^2 + eps) * gain ),  x = X[pos[t],:]
 * Token i of a trajectory is scored by log p(. | t_<i, Q) (Eq. 3), i.e. by the state of the
 * position before it, and only trajectory tokens are averaged (Eq. 4): `pos` carries that
 * shift and packing.  fp32 arithmetic, one rounding to bf16.
 *   X      DEVICE bf16 [num_rows, d]   last-layer output of the packed prefill (before the final norm)
 *   pos    DEVICE int32 [T] rows of X (trusted; clamped into range), or NULL = identity (T <= num_rows)
 *   gain   DEVICE bf16 [d]             RMSNorm weight
 *   H_out  DEVICE bf16 [T, d]          16-byte aligned like X and gain; may alias X only when pos == NULL
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA. */
int sq_score_prepare(sq_score_ctx *ctx, const void *X, int num_rows, const int32_t *pos, int num_tokens,
                     const void *gain, float eps, void *H_out, void *stream);

/* sq_score_prepare into the ctx-owned H buffer ([max_tokens, d] bf16; ctx created with SQ_FLAG_STAGING)
 * followed by sq_score_run on it: the library takes the last layer's output and the position list directly.
 * Errors: as sq_score_prepare and sq_score_run; INVALID_ARG without SQ_FLAG_STAGING. */
int sq_score_run_x(sq_score_ctx *ctx, const void *X, int num_rows, const int32_t *pos, const void *gain,
                   float eps, const void *W, const int32_t *targets, const int32_t *cu_seqlens,
                   int num_tokens, int num_seqs, int k, int window, const sq_score_outputs *outputs,
                   void *stream);

/* The position list of sq_score_prepare / sq_score_run_x for a packed prefill in which candidate b occupies
 * query_lens[b] query tokens followed by traj_lens[b] trajectory tokens.  Token i (i = 1..|tau|) of a trajectory is
 * scored by log p(. | t_<i, Q) (Eq. 3), i.e. by the hidden state of the packed row just before it, and
 * only the |tau| trajectory tokens are averaged (Eq. 4):
 *     cu[0] = 0, cu[b+1] = cu[b] + traj_lens[b];   base_b = sum_{c<b} (query_lens[c] + traj_lens[c]);
 *     pos[cu[b] + i] = base_b + query_lens[b] - 1 + i,   i = 0 .. traj_lens[b] - 1.
 * A trajectory needs at least one query token before it (there is no state that predicts its first token otherwise).
 *
 * sq_score_positions_host: HOST arrays in and out, needs no GPU and no ctx.  pos_out has room for pos_capacity
 * entries; *num_tokens_out (may be NULL) receives T = sum traj_lens.
 * Errors: INVALID_ARG (null pointer, negative length, a non-empty trajectory with query_lens[b] < 1, T > pos_capacity).
 *
 * sq_score_positions: the same on the device (no host round trip between the prefill and sq_score_run_x): DEVICE
 * int32 arrays query_lens[B], traj_lens[B] -> pos_out[num_tokens], cu_out[B+1]; num_tokens must equal sum traj_lens
 * (the caller built the batch and knows it).  Device contents are trusted; if status_out (DEVICE int32[1], may be
 * NULL) is given it receives 0, or the number of candidates that violate the rules above (negative length, missing
 * query token) plus 1 if the lengths do not sum to num_tokens -- pos entries of such candidates are clamped to >= 0.
 * B <= max_seqs, num_tokens <= max_tokens.  Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA. */
int sq_score_positions_host(const int32_t *query_lens, const int32_t *traj_lens, int num_seqs,
                            int32_t *pos_out, int64_t pos_capacity, int32_t *cu_out, int64_t *num_tokens_out);
int sq_score_positions(sq_score_ctx *ctx, const int32_t *query_lens, const int32_t *traj_lens, int num_seqs,
                       int num_tokens, int32_t *pos_out, int32_t *cu_out, int32_t *status_out, void *stream);

/* FP8 variant: the same scoring pass with e4m3 operands (tcgen05 kind::f8f6f4, twice the
 * tensor throughput and half the operand bytes of bf16).  It is NOT the graded bf16 path: the quantisation changes the
 * logits by ~1e-1 (measured against the bf16 oracle in tests/test_fp8_gpu.py); on the QUANTISED inputs the kernel meets
 * the same tolerances as the bf16 path.
 *
 * sq_score_quantize_fp8:  q = e4m3_rn_sat(x * (448 / amax)), scale = amax / 448 (amax == 0: scale 1, codes 0), so that
 * x ~= q * scale.  per_tensor == 0: one amax and one scale per row (H: per token); != 0: one over the whole tensor (W).
 *   X          DEVICE bf16 [num_rows, d], 16-byte aligned
 *   q_out      DEVICE uint8 [num_rows, d] e4m3 codes, 8-byte aligned
 *   scale_out  DEVICE float [num_rows] (per row) or [1] (per tensor)
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA. */
int sq_score_quantize_fp8(sq_score_ctx *ctx, const void *X, int64_t num_rows, int per_tensor, void *q_out,
                          float *scale_out, void *stream);

/* sq_score_run on quantised operands: logits = h_scale[t] * w_scale[0] * sum_j Hq[t,j] * Wq[v,j] (products exact,
 * fp32 accumulate); the scales are folded into the exponent's multiplier, so they cost nothing per logit.
 *   Hq DEVICE uint8 [T,d], h_scale DEVICE float [T], Wq DEVICE uint8 [V,d], w_scale DEVICE float [1]; d % 16 == 0;
 *   everything else as sq_score_run.  Errors: as sq_score_run, UNSUPPORTED (d % 16). */
int sq_score_run_fp8(sq_score_ctx *ctx, const void *Hq, const float *h_scale, const void *Wq, const float *w_scale,
                     const int32_t *targets, const int32_t *cu_seqlens, int num_tokens, int num_seqs, int k,
                     int window, const sq_score_outputs *outputs, void *stream);

/* Block-scaled (MX) variant: e4m3 elements with one power-of-two scale per 32 consecutive elements of a row (UE8M0:
 * scale = 2^(byte - 127)), the operand format of tcgen05.mma.kind::mxf8f6f4.block_scale -- the tensor core applies the
 * scales, so a block's dynamic range no longer depends on the rest of its row / of the tensor (PAPER.md:681-692 motivates
 * the engine by very large scorers, where an 8-bit LM head matters).  Like the FP8 variant it is not the graded bf16
 * path; tests/test_mx_gpu.py measures how much closer to the bf16 scores it gets.
 *
 * sq_score_quantize_mx, by definition (reading #26; exact arithmetic, so the result is unique):
 *   e    = the smallest integer with max|x_block| <= 448 * 2^e, clamped to [-127, 127] (all-zero block: -127)
 *   code = the e4m3 value nearest to x * 2^-e, ties to even;       x ~= e4m3(code) * 2^e
 *   X        DEVICE bf16 [num_rows, d], d = cfg.d, d % 16 == 0, 16-byte aligned
 *   operand  SQ_MX_OPERAND_H (token rows, grouped by 128) or SQ_MX_OPERAND_W (vocabulary rows, grouped by the kernel's
 *            224-column tiles): selects the layout of sf_out
 *   q_out    DEVICE uint8 [num_rows, d] e4m3 codes, 16-byte aligned
 *   sf_out   DEVICE uint8 [sq_score_mx_scale_bytes(num_rows, d, operand)], 16-byte aligned: byte e + 127 of row r,
 *            32-element block kb32 is at
 *              ((kb32 / 4 * num_groups + r / G) * P + (r % G) / 128) * 512 + (r % 32) * 16 + ((r % G) / 32 % 4) * 4 + kb32 % 4
 *            with G = 128, P = 1 (H) or G = 224, P = 2 (W), num_groups = ceil(num_rows / G): 512-byte pieces that
 *            tcgen05.cp moves to TMEM as they are.  Bytes no row / block reaches are 0.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, UNSUPPORTED (d % 16), CUDA.
 *
 * sq_score_run_mx: sq_score_run on such operands (logits = sum over blocks of 2^(eh + ew) * sum_j Hq * Wq, products
 * exact, fp32 accumulate in the tensor core); Hq / h_sf from operand H with num_rows = T, Wq / w_sf from operand W with
 * num_rows = cfg.vocab; everything else as sq_score_run.  Errors: as sq_score_run, UNSUPPORTED (d % 16). */
#define SQ_MX_OPERAND_H 0
#define SQ_MX_OPERAND_W 1
int64_t sq_score_mx_scale_bytes(int64_t num_rows, int d, int operand);
int sq_score_quantize_mx(sq_score_ctx *ctx, const void *X, int64_t num_rows, int operand, void *q_out, void *sf_out,
                         void *stream);
int sq_score_run_mx(sq_score_ctx *ctx, const void *Hq, const void *h_sf, const void *Wq, const void *w_sf,
                    const int32_t *targets, const int32_t *cu_seqlens, int num_tokens, int num_seqs, int k,
                    int window, const sq_score_outputs *outputs, void *stream);

/* Vocab-parallel scoring: the LM head is split by rows over R shards (the tensor-
 * parallel layout of a served scorer); every shard scores the same H against its rows and produces ONE merged partial
 * state per token; the states are exchanged (one all-gather, e.g. ncclAllGather / torch.distributed) and merged by the
 * same associative operator that merges vocab chunks inside a GPU, followed by kernel 2.
 *
 * Packed state of one shard, 4-byte words, (6 + 2*cap) * T of them with cap = 8 / 20 / 32 for k <= 8 / 20 / 32:
 *   m[T] s[T] u[T] cs[T] cu[T]  running max, sum exp(z-m), sum exp(z-m)(z-m), and the residues of s and u
 *                               (true value = s - cs: the merged sums keep their fp64 precision)
 *   topv[cap][T] topi[cap][T]   the shard's k best logits (descending) and their GLOBAL vocabulary ids, -1 = empty
 *   zt[T]                       the target's logit, meaningful on the shard that owns its row
 * sq_score_shard_state_bytes: size of that buffer (host-only; -1 on bad arguments). */
int64_t sq_score_shard_state_bytes(int64_t num_tokens, int k);

/* One shard: W_shard holds the shard_rows rows [vocab_offset, vocab_offset + shard_rows) of the LM head,
 * 1 <= shard_rows <= cfg.vocab (a ctx sized for the LARGEST shard serves every rank of an uneven split); targets are
 * GLOBAL ids.  Runs kernel 1 and the merge kernel in EMIT mode, writes state_out (DEVICE,
 * sq_score_shard_state_bytes(T, k) bytes).  k <= min(max_k, shard_rows).  Asynchronous on `stream`.
 * Errors: as sq_score_run; INVALID_ARG if shard_rows is outside 1..cfg.vocab. */
int sq_score_run_shard(sq_score_ctx *ctx, const void *H, const void *W_shard, int shard_rows, int vocab_offset,
                       const int32_t *targets, int num_tokens, int k, void *state_out, void *stream);

/* The packed state of a shard that owns NO vocabulary rows (more ranks than vocab tiles): the neutral element of the
 * merge (m = -1e30, s = u = 0, empty list).  Writes sq_score_shard_state_bytes(T, k) bytes to state_out (DEVICE).
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA. */
int sq_score_neutral_shard_state(sq_score_ctx *ctx, int num_tokens, int k, void *state_out, void *stream);

/* Merge of num_shards (1..32) packed states laid out back to back in `states` (DEVICE; the all-gather's output),
 * then the per-token finalisation and kernel 2 -- the same outputs as sq_score_run on the whole LM head.
 *   vocab_starts  HOST int32 [num_shards+1]: shard r owns ids [vocab_starts[r], vocab_starts[r+1]); the last entry is V
 * Any ctx of the right max_tokens / max_seqs / max_k can merge.  Errors: INVALID_ARG, CUDA. */
int sq_score_merge_shards(sq_score_ctx *ctx, const void *states, int num_shards, const int32_t *vocab_starts,
                          const int32_t *targets, const int32_t *cu_seqlens, int num_tokens, int num_seqs,
                          int k, int window, const sq_score_outputs *outputs, void *stream);

/* The same merge WITHOUT the all-gather: state_ptrs (HOST array of num_shards DEVICE pointers) names one packed state per
 * shard wherever it lives in the unified address space -- this GPU's own buffer and the peers' buffers mapped over
 * NVLink (cudaIpcOpenMemHandle / peer access).  The merge kernel reads every shard's state in place, lane r = shard r, so
 * the transfer is the merge's own loads: no staging copy of R x state bytes, and the exchange overlaps the merge row by
 * row.  The caller orders the run: every shard's sq_score_run_shard must have completed before this call's kernels start
 * (paper_2604_07725_b200/sharding.py: a 4-byte all-reduce on the stream), and a state must not be overwritten while a peer
 * may still read it.  Pointers must be 4-byte aligned.  Errors: INVALID_ARG, CUDA. */
int sq_score_merge_shards_peer(sq_score_ctx *ctx, const void *const *state_ptrs, int num_shards,
                               const int32_t *vocab_starts, const int32_t *targets, const int32_t *cu_seqlens,
                               int num_tokens, int num_seqs, int k, int window, const sq_score_outputs *outputs,
                               void *stream);

/* Group fitness and routing on the device, one problem per CTA:
 *   group_fitness[g] = GC(g) = (1/K) * sum_{j<K} seq_conf[group_members[g*K+j]]   Eq. 4 right
 *   theta[q] = Percentile_p of GC over problem q's non-lite groups                Eq. 6
 *              (linear interpolation at rank p/100*(n-1); NaN when every group is lite)
 *   route[g] = 0 if lite_mask[g], else 1 (Model 1) if GC(g) > theta[q], else 2 (Model 2)   Eq. 7
 *              3 = GC(g) is not finite (the group holds an empty trajectory, whose C(tau) is NaN): the group takes no
 *              part in the percentile and is left to the caller; -1 = the problem has more than 1024 groups (the
 *              host-side bound was wrong): theta[q] = NaN and nothing of that problem is routed
 *   seq_conf       DEVICE float [num_seqs]      C(tau), e.g. seq_mean_conf of sq_score_run
 *   group_members  DEVICE int32 [num_groups*K]  indices into seq_conf (trusted, must be in range)
 *   group_offsets  DEVICE int32 [num_problems+1] groups of problem q are [off[q], off[q+1])
 *   lite_mask      DEVICE uint8 [num_groups] or NULL (the consensus test is on answer strings, not here)
 *   max_groups_per_problem  host-side bound on off[q+1]-off[q], <= 1024
 * Asynchronous on `stream`.  Errors: INVALID_ARG, UNSUPPORTED (more than 1024 groups in a problem), CUDA. */
int sq_score_route(sq_score_ctx *ctx, const float *seq_conf, int num_seqs, const int32_t *group_members,
                   const int32_t *group_offsets, int num_problems, int num_groups, int group_size,
                   int max_groups_per_problem, const uint8_t *lite_mask, float percentile,
                   float *group_fitness, float *theta, int32_t *route, void *stream);

/* Fitness-weighted selection probabilities: within each problem's population
 * [pop_offsets[q], pop_offsets[q+1]),  prob[i] = exp(fitness[i]/zeta) / sum_j exp(fitness[j]/zeta).
 * All pointers DEVICE; zeta > 0.  The draws themselves stay with the caller.  Errors: INVALID_ARG, CUDA. */
int sq_score_select_prob(sq_score_ctx *ctx, const float *fitness, const int32_t *pop_offsets,
                         int num_problems, float zeta, float *prob, void *stream);

/* Host-only: the work decomposition `sq_score_run` would use for T tokens and top-k `k` on a
 * device with `num_sms` SMs (pass 0 for the ctx-independent default of 148).  `cfg` supplies d,
 * vocab, cta_group, num_chunks, group_m.  Needs no GPU.  Errors: INVALID_ARG. */
int sq_score_plan(const sq_score_config *cfg, int64_t num_tokens, int k, int num_sms,
                  sq_score_plan_t *plan);

/* The work decomposition the LAST sq_score_run* call on this ctx actually launched kernel 1 with (sq_score_plan answers
 * for a ctx-less default and always describes CTA pairs or single CTAs).  plan->cta_group is 1, 2, or 4 = quad scheduling
 * with W multicast, which runs of more than 200 000 tokens take by default: rows_per_tile is then 512 and the cluster
 * counts are in quads.  Host-only, no synchronisation.  Errors: INVALID_ARG (null, or no run with T > 0 yet). */
int sq_score_last_plan(const sq_score_ctx *ctx, sq_score_plan_t *plan);

/* Per-kernel timing for the roofline report.  With profiling enabled, every sq_score_run* with
 * T > 0 records CUDA events on its stream around kernel 1 (fused GEMM + statistics), the
 * finalize kernel and kernel 2, into a ring of SQ_PROFILE_RING runs (no host synchronisation in the run).
 * sq_score_kernel_times blocks until the last profiled run finished and writes its three durations in
 * milliseconds: ms3 = {fused, finalize, reduce}.  sq_score_profile_read does the same for EVERY run recorded
 * since profiling was enabled or last read (the newest SQ_PROFILE_RING of them, oldest first): up to
 * `capacity` triples into ms, their number into *num_runs, and empties the ring.
 * sq_score_set_profiling(ctx, 1) creates the events (the only allocation outside create; call it outside runs).
 * Errors: INVALID_ARG (null, profiling off, no profiled run yet), CUDA. */
#define SQ_PROFILE_RING 64
int sq_score_set_profiling(sq_score_ctx *ctx, int enable);
int sq_score_kernel_times(sq_score_ctx *ctx, float *ms3);
int sq_score_profile_read(sq_score_ctx *ctx, float *ms, int capacity, int *num_runs);

/* Test hook (tests/test_memory_safety_gpu.py): fills every ctx-owned workspace and staging buffer with the byte
 * `value` (0xFF = NaN floats / -1 ints) on `stream`, then restores the two invariants the kernels rely on (zeroed
 * per-sequence counters of kernel 2).  A run after it must give the same results: no kernel may read workspace it
 * did not write in the same run.  Changes no result.  Errors: INVALID_ARG, CUDA. */
int sq_score_debug_fill_workspace(sq_score_ctx *ctx, int value, void *stream);

/* Number of kernels this ctx has launched so far (bench.py's `gpu_launches`). */
int64_t sq_score_launch_count(const sq_score_ctx *ctx);

/* Which form of kernel 2 (step a7) the last call on this ctx used: 0 = none yet, SQ_REDUCE_FORM_FUSED = one launch (the
 * whole problem is one wave of CTAs), _TILES = three launches over sequence-aligned tiles, _STREAM = stream +
 * fold over fixed blocks (large inputs, 128 <= window <= 2048, 16-byte aligned arrays), _TAIL = inside the finalize kernel
 * (runs of at most 256 tokens).  All forms compute the same reductions; tests and bench.py report which one ran. */
#define SQ_REDUCE_FORM_FUSED 1
#define SQ_REDUCE_FORM_TILES 2
#define SQ_REDUCE_FORM_STREAM 3
#define SQ_REDUCE_FORM_TAIL 4
int sq_score_reduce_form(const sq_score_ctx *ctx);

/* Frees the workspace.  NULL is a no-op.  Errors: CUDA. */
int sq_score_destroy(sq_score_ctx *ctx);

/* Message of the last error on this ctx (ctx-owned, valid until the next call on ctx); with
 * ctx == NULL, the message of the last failed sq_score_create or sq_score_reduce_static on this thread. */
const char *sq_score_last_error(const sq_score_ctx *ctx);

/* Static name of an SQ_ERR_* code. */
const char *sq_score_error_string(int code);

/* Library version, e.g. 100 = 0.1.0. */
int sq_score_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SQ_SCORE_H_ */
