"""ctypes binding with the same names as the C ABI (include/sq_score.h)."""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

from . import build as _build

SQ_MAX_K = 32
SQ_MAX_CHUNKS = 160
SQ_PROFILE_RING = 64
FLAG_REDUCE_ONLY = 1
FLAG_STAGING = 2
STATIC_MAX_TOKENS = 1 << 22     # SQ_STATIC_MAX_TOKENS / SQ_STATIC_MAX_SEQS: limits of reduce_static
STATIC_MAX_SEQS = 4096
MX_OPERAND_H, MX_OPERAND_W = 0, 1
ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_NOMEM = -1, -2, -3, -4


class sq_score_config(C.Structure):
    _fields_ = [("device", C.c_int), ("d", C.c_int), ("vocab", C.c_int), ("max_tokens", C.c_int64),
                ("max_seqs", C.c_int), ("max_k", C.c_int), ("cta_group", C.c_int), ("num_chunks", C.c_int),
                ("group_m", C.c_int), ("flags", C.c_int), ("wait_seconds", C.c_int),
                ("debug_flags", C.c_int), ("cluster4", C.c_int), ("region_mult", C.c_int)]


class sq_score_outputs(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in
                ("lse", "target_logprob", "entropy", "conf", "topk_logprob", "topk_index",
                 "seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")]


class sq_score_plan_t(C.Structure):
    _fields_ = [(n, C.c_int) for n in
                ("cta_group", "rows_per_tile", "m_tiles", "num_vtiles", "num_k_blocks", "num_chunks", "chunks_per_gang",
                 "tiles_per_chunk", "num_units", "num_clusters", "num_gangs", "gang_size", "gangs_big", "clusters_used",
                 "max_batches", "topk_cap")] + [("chunk_vtile", C.c_int * (SQ_MAX_CHUNKS + 1))]


class SqScoreError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("sq_score error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Loads csrc/libsq_score.so, rebuilding it first when a source is newer.  Fails loudly if it cannot be built or
    loaded: a stale library is never used in place of one that failed to build."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.is_stale():
        path = _build.build()      # raises with nvcc's output
    L = C.CDLL(path)
    L.sq_score_create.argtypes = [C.POINTER(sq_score_config), C.POINTER(C.c_void_p)]
    L.sq_score_create.restype = C.c_int
    L.sq_score_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                               C.c_int, C.c_int, C.POINTER(sq_score_outputs), C.c_void_p]
    L.sq_score_run.restype = C.c_int
    L.sq_score_run_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                    C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    L.sq_score_run_host.restype = C.c_int
    L.sq_score_reduce.argtypes = [C.c_void_p] + [C.c_void_p] * 5 + [C.c_int64, C.c_int, C.c_int] + [C.c_void_p] * 5
    L.sq_score_reduce.restype = C.c_int
    L.sq_score_reduce_static.argtypes = [C.c_void_p] * 5 + [C.c_int64, C.c_int, C.c_int, C.c_int] + [C.c_void_p] * 5
    L.sq_score_reduce_static.restype = C.c_int
    L.sq_score_route.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int,
                                 C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.sq_score_route.restype = C.c_int
    L.sq_score_select_prob.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_float, C.c_void_p, C.c_void_p]
    L.sq_score_select_prob.restype = C.c_int
    L.sq_score_prepare.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p]
    L.sq_score_prepare.restype = C.c_int
    L.sq_score_run_x.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p,
                                 C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(sq_score_outputs), C.c_void_p]
    L.sq_score_run_x.restype = C.c_int
    L.sq_score_shard_state_bytes.argtypes = [C.c_int64, C.c_int]
    L.sq_score_shard_state_bytes.restype = C.c_int64
    L.sq_score_run_shard.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    L.sq_score_run_shard.restype = C.c_int
    L.sq_score_neutral_shard_state.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    L.sq_score_neutral_shard_state.restype = C.c_int
    L.sq_score_positions_host.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_int, C.POINTER(C.c_int32), C.c_int64,
                                          C.POINTER(C.c_int32), C.POINTER(C.c_int64)]
    L.sq_score_positions_host.restype = C.c_int
    L.sq_score_positions.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.sq_score_positions.restype = C.c_int
    L.sq_score_debug_fill_workspace.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
    L.sq_score_debug_fill_workspace.restype = C.c_int
    L.sq_score_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_int)]
    L.sq_score_profile_read.restype = C.c_int
    L.sq_score_merge_shards.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_int32), C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                        C.c_int, C.c_int, C.POINTER(sq_score_outputs), C.c_void_p]
    L.sq_score_merge_shards.restype = C.c_int
    L.sq_score_quantize_fp8.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    L.sq_score_quantize_fp8.restype = C.c_int
    L.sq_score_merge_shards_peer.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                             C.c_int, C.c_int, C.POINTER(sq_score_outputs), C.c_void_p]
    L.sq_score_merge_shards_peer.restype = C.c_int
    L.sq_score_run_fp8.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                   C.c_int, C.c_int, C.POINTER(sq_score_outputs), C.c_void_p]
    L.sq_score_run_fp8.restype = C.c_int
    L.sq_score_mx_scale_bytes.argtypes = [C.c_int64, C.c_int, C.c_int]
    L.sq_score_mx_scale_bytes.restype = C.c_int64
    L.sq_score_quantize_mx.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    L.sq_score_quantize_mx.restype = C.c_int
    L.sq_score_run_mx.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                  C.c_int, C.c_int, C.POINTER(sq_score_outputs), C.c_void_p]
    L.sq_score_run_mx.restype = C.c_int
    L.sq_score_plan.argtypes = [C.POINTER(sq_score_config), C.c_int64, C.c_int, C.c_int, C.POINTER(sq_score_plan_t)]
    L.sq_score_plan.restype = C.c_int
    L.sq_score_set_profiling.argtypes = [C.c_void_p, C.c_int]
    L.sq_score_set_profiling.restype = C.c_int
    L.sq_score_kernel_times.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    L.sq_score_kernel_times.restype = C.c_int
    L.sq_score_launch_count.argtypes = [C.c_void_p]
    L.sq_score_launch_count.restype = C.c_int64
    L.sq_score_last_plan.argtypes = [C.c_void_p, C.POINTER(sq_score_plan_t)]
    L.sq_score_last_plan.restype = C.c_int
    L.sq_score_reduce_form.argtypes = [C.c_void_p]
    L.sq_score_reduce_form.restype = C.c_int
    L.sq_score_destroy.argtypes = [C.c_void_p]
    L.sq_score_destroy.restype = C.c_int
    L.sq_score_last_error.argtypes = [C.c_void_p]
    L.sq_score_last_error.restype = C.c_char_p
    L.sq_score_error_string.argtypes = [C.c_int]
    L.sq_score_error_string.restype = C.c_char_p
    L.sq_score_version.argtypes = []
    L.sq_score_version.restype = C.c_int
    _lib = L
    return L


def version() -> int:
    return lib().sq_score_version()


def plan(d: int, vocab: int, num_tokens: int, k: int, num_sms: int = 0, cta_group: int = 0,
         num_chunks: int = 0, group_m: int = 0) -> Dict[str, int]:
    """sq_score_plan: host-only work decomposition (no GPU needed)."""
    cfg = sq_score_config(0, d, vocab, max(1, num_tokens), 1, max(1, min(k, SQ_MAX_K)), cta_group, num_chunks, group_m, 0, 0)
    out = sq_score_plan_t()
    rc = lib().sq_score_plan(C.byref(cfg), num_tokens, k, num_sms, C.byref(out))
    if rc != 0:
        raise SqScoreError(rc, lib().sq_score_error_string(rc).decode())
    res = {n: getattr(out, n) for n, _ in sq_score_plan_t._fields_ if n != "chunk_vtile"}
    res["chunk_vtile"] = list(out.chunk_vtile[: out.num_chunks + 1])
    return res


def shard_state_bytes(num_tokens: int, k: int) -> int:
    """sq_score_shard_state_bytes (host-only)."""
    n = lib().sq_score_shard_state_bytes(num_tokens, k)
    if n < 0:
        raise SqScoreError(ERR_INVALID_ARG, "bad num_tokens / k")
    return n


def reduce_static(target_logprob, entropy, conf, cu_seqlens, window: int, targets=None, vocab: int = 1,
                  out: Optional[dict] = None, stream=None) -> dict:
    """sq_score_reduce_static: kernel 2 without a ctx, for callers that cannot allocate device memory (a plug-in inside a
    serving engine whose pool already owns the free HBM; a latency-critical loop that cannot afford cudaMalloc's
    device-wide synchronisation).  The library allocates nothing: its scratch is a fixed array in the device image, so at
    most STATIC_MAX_TOKENS tokens and STATIC_MAX_SEQS sequences per call, and calls that may overlap on the GPU race on
    it -- keep them on one stream.  Pass `out` (the four float32 [B] tensors of SqScore.reduce) to keep this wrapper
    from allocating too; without it the result tensors come from torch's allocator.  Runs on the tensors' device."""
    import torch
    B = cu_seqlens.shape[0] - 1
    if out is None:
        out = {n: torch.empty(B, dtype=torch.float32, device=conf.device)
               for n in ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")}
    L = lib()
    with torch.cuda.device(conf.device):          # the call uses the thread's current device
        s = stream if stream is not None else torch.cuda.current_stream()
        rc = L.sq_score_reduce_static(_ptr(target_logprob), _ptr(entropy), _ptr(conf), _ptr(targets), _ptr(cu_seqlens),
                                      conf.shape[0], B, vocab, window, _ptr(out["seq_mean_logprob"]),
                                      _ptr(out["seq_mean_entropy"]), _ptr(out["seq_mean_conf"]),
                                      _ptr(out["seq_min_window_conf"]), s.cuda_stream)
    if rc != 0:
        raise SqScoreError(rc, L.sq_score_last_error(None).decode())
    return out


def shard_vocab(vocab: int, world_size: int, multiple: int = 256) -> List[int]:
    """Row split of the LM head for vocab-parallel scoring: world_size contiguous shards, sizes a multiple of
    `multiple` rows (one vocab tile) except the last, as equal as that allows.  Returns the world_size + 1 starts."""
    tiles = -(-vocab // multiple)
    starts = [min(vocab, (tiles * r // world_size) * multiple) for r in range(world_size)]
    return starts + [vocab]


def _ptr(t) -> Optional[int]:
    return None if t is None else t.data_ptr()


class SqScore:
    """sq_score_create / sq_score_run / sq_score_destroy on torch tensors (device memory + streams)."""

    def __init__(self, d: int, vocab: int, max_tokens: int, max_seqs: int, max_k: int = 20, device: int = 0,
                 cta_group: int = 0, num_chunks: int = 0, group_m: int = 0, reduce_only: bool = False,
                 staging: bool = False, wait_seconds: int = 0, debug_flags: int = 0, cluster4: int = 0, region_mult: int = 0):
        """`staging=True` (SQ_FLAG_STAGING) also allocates what run_host / run_x need; no run* call ever allocates.
        `debug_flags` (SQ_DEBUG_* bits), `cluster4` and `region_mult` choose between code paths with the same results
        (include/sq_score.h); tests force each path through them."""
        self._L = lib()
        self.cfg = sq_score_config(device, d, vocab, max_tokens, max_seqs, max_k, cta_group, num_chunks, group_m,
                                   (FLAG_REDUCE_ONLY if reduce_only else 0) | (FLAG_STAGING if staging else 0), wait_seconds,
                                   int(debug_flags or 0), cluster4, region_mult)
        h = C.c_void_p()
        rc = self._L.sq_score_create(C.byref(self.cfg), C.byref(h))
        if rc != 0:
            raise SqScoreError(rc, self._L.sq_score_last_error(None).decode())
        self._h = h
        self.device = device

    def _check(self, rc: int):
        if rc != 0:
            raise SqScoreError(rc, self._L.sq_score_last_error(self._h).decode())

    @staticmethod
    def _stream(stream) -> int:
        import torch
        s = stream if stream is not None else torch.cuda.current_stream()
        return s.cuda_stream

    def run(self, H, W, targets, cu_seqlens, k: int, window: int, stream=None, per_token: bool = True,
            topk: bool = True, out: Optional[dict] = None) -> dict:
        """sq_score_run.  Allocates (or reuses `out`) the output tensors; asynchronous on the stream."""
        import torch
        T, B = H.shape[0], cu_seqlens.shape[0] - 1
        dev = H.device
        if out is None:
            out = self._alloc_out(T, B, k, dev, per_token, topk)
        o = sq_score_outputs(*[_ptr(out.get(n)) for n, _ in sq_score_outputs._fields_])
        self._check(self._L.sq_score_run(self._h, _ptr(H), _ptr(W), _ptr(targets), _ptr(cu_seqlens), T, B, k, window,
                                         C.byref(o), self._stream(stream)))
        return out

    def _alloc_out(self, T, B, k, dev, per_token, topk):
        import torch
        out = {}
        f = dict(dtype=torch.float32, device=dev)
        if per_token:
            for n in ("lse", "target_logprob", "entropy", "conf"):
                out[n] = torch.empty(T, **f)
        if topk:
            out["topk_logprob"] = torch.empty(T, k, **f)
            out["topk_index"] = torch.empty(T, k, dtype=torch.int32, device=dev)
        for n in ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf"):
            out[n] = torch.empty(B, **f)
        return out

    def prepare(self, X, pos, gain, eps: float, out=None, stream=None):
        """sq_score_prepare: H[t] = bf16(RMSNorm(X[pos[t]]) * gain); pos None = identity."""
        import torch
        T = X.shape[0] if pos is None else pos.shape[0]
        if out is None:
            out = torch.empty(T, X.shape[1], dtype=torch.bfloat16, device=X.device)
        self._check(self._L.sq_score_prepare(self._h, _ptr(X), X.shape[0], _ptr(pos), T, _ptr(gain), float(eps), _ptr(out),
                                             self._stream(stream)))
        return out

    def run_x(self, X, pos, gain, eps: float, W, targets, cu_seqlens, k: int, window: int, stream=None,
              per_token: bool = True, topk: bool = True, out: Optional[dict] = None) -> dict:
        """sq_score_run_x: prepare (gather + final RMSNorm) into the ctx's H buffer, then sq_score_run."""
        T = X.shape[0] if pos is None else pos.shape[0]
        B = cu_seqlens.shape[0] - 1
        if out is None:
            out = self._alloc_out(T, B, k, X.device, per_token, topk)
        o = sq_score_outputs(*[_ptr(out.get(n)) for n, _ in sq_score_outputs._fields_])
        self._check(self._L.sq_score_run_x(self._h, _ptr(X), X.shape[0], _ptr(pos), _ptr(gain), float(eps), _ptr(W), _ptr(targets),
                                           _ptr(cu_seqlens), T, B, k, window, C.byref(o), self._stream(stream)))
        return out

    def run_shard(self, H, W_shard, vocab_offset: int, targets, k: int, out=None, stream=None):
        """sq_score_run_shard: the rows W_shard of the LM head (at most the ctx's vocab of them) -> packed partial state
        (a float32 tensor of shard_state_bytes(T, k) / 4 words; ids inside are int32 bit patterns)."""
        import torch
        T = H.shape[0]
        if out is None:
            out = torch.empty(shard_state_bytes(T, k) // 4, dtype=torch.float32, device=H.device)
        self._check(self._L.sq_score_run_shard(self._h, _ptr(H), _ptr(W_shard), W_shard.shape[0], int(vocab_offset), _ptr(targets),
                                               T, k, _ptr(out), self._stream(stream)))
        return out

    def neutral_shard_state(self, num_tokens: int, k: int, device=None, out=None, stream=None):
        """sq_score_neutral_shard_state: the packed state of a shard that owns no vocabulary rows."""
        import torch
        if out is None:
            out = torch.empty(shard_state_bytes(num_tokens, k) // 4, dtype=torch.float32,
                              device=device if device is not None else torch.device("cuda", self.device))
        self._check(self._L.sq_score_neutral_shard_state(self._h, num_tokens, k, _ptr(out), self._stream(stream)))
        return out

    def positions(self, query_lens, traj_lens, num_tokens: int, stream=None, with_status: bool = False):
        """sq_score_positions: device int32 [B] query / trajectory lengths -> (pos [num_tokens], cu_seqlens [B+1]) on the
        device, no host round trip; `num_tokens` = sum of traj_lens (known to the caller)."""
        import torch
        B = traj_lens.shape[0]
        dev = traj_lens.device
        pos = torch.empty(num_tokens, dtype=torch.int32, device=dev)
        cu = torch.empty(B + 1, dtype=torch.int32, device=dev)
        status = torch.empty(1, dtype=torch.int32, device=dev) if with_status else None
        self._check(self._L.sq_score_positions(self._h, _ptr(query_lens), _ptr(traj_lens), B, num_tokens, _ptr(pos), _ptr(cu),
                                               _ptr(status), self._stream(stream)))
        return (pos, cu, status) if with_status else (pos, cu)

    def merge_shards(self, states, vocab_starts: Sequence[int], targets, cu_seqlens, k: int, window: int, stream=None,
                     per_token: bool = True, topk: bool = True, out: Optional[dict] = None) -> dict:
        """sq_score_merge_shards: `states` is the [R, words] tensor the all-gather produced."""
        R = len(vocab_starts) - 1
        T, B = targets.shape[0], cu_seqlens.shape[0] - 1
        if out is None:
            out = self._alloc_out(T, B, k, targets.device, per_token, topk)
        o = sq_score_outputs(*[_ptr(out.get(n)) for n, _ in sq_score_outputs._fields_])
        vs = (C.c_int32 * (R + 1))(*[int(v) for v in vocab_starts])
        self._check(self._L.sq_score_merge_shards(self._h, _ptr(states), R, vs, _ptr(targets), _ptr(cu_seqlens), T, B, k, window,
                                                  C.byref(o), self._stream(stream)))
        return out

    def merge_shards_peer(self, states: Sequence, vocab_starts: Sequence[int], targets, cu_seqlens, k: int, window: int, stream=None,
                          per_token: bool = True, topk: bool = True, out: Optional[dict] = None) -> dict:
        """sq_score_merge_shards_peer: `states` is a list of R tensors (or raw device addresses), one packed state per
        shard, read in place -- peers' buffers included."""
        R = len(vocab_starts) - 1
        if len(states) != R:
            raise ValueError("%d states for %d shards" % (len(states), R))
        T, B = targets.shape[0], cu_seqlens.shape[0] - 1
        if out is None:
            out = self._alloc_out(T, B, k, targets.device, per_token, topk)
        o = sq_score_outputs(*[_ptr(out.get(n)) for n, _ in sq_score_outputs._fields_])
        vs = (C.c_int32 * (R + 1))(*[int(v) for v in vocab_starts])
        ptrs = (C.c_void_p * R)(*[(st if isinstance(st, int) else st.data_ptr()) for st in states])
        self._check(self._L.sq_score_merge_shards_peer(self._h, ptrs, R, vs, _ptr(targets), _ptr(cu_seqlens), T, B, k, window,
                                                       C.byref(o), self._stream(stream)))
        return out

    def quantize_fp8(self, X, per_tensor: bool, stream=None, out=None):
        """sq_score_quantize_fp8: bf16 [rows, d] -> (uint8 e4m3 codes [rows, d], float32 scales [rows] or [1]);
        `out` = (codes, scales) reuses the tensors of an earlier call."""
        import torch
        rows = X.shape[0]
        if out is not None:
            q, scale = out
        else:
            q = torch.empty(rows, X.shape[1], dtype=torch.uint8, device=X.device)
            scale = torch.empty(1 if per_tensor else rows, dtype=torch.float32, device=X.device)
        self._check(self._L.sq_score_quantize_fp8(self._h, _ptr(X), rows, 1 if per_tensor else 0, _ptr(q), _ptr(scale),
                                                  self._stream(stream)))
        return q, scale

    def run_fp8(self, Hq, h_scale, Wq, w_scale, targets, cu_seqlens, k: int, window: int, stream=None, per_token: bool = True,
                topk: bool = True, out: Optional[dict] = None) -> dict:
        """sq_score_run_fp8: the scoring pass on e4m3 operands with per-token / per-tensor scales."""
        T, B = Hq.shape[0], cu_seqlens.shape[0] - 1
        if out is None:
            out = self._alloc_out(T, B, k, Hq.device, per_token, topk)
        o = sq_score_outputs(*[_ptr(out.get(n)) for n, _ in sq_score_outputs._fields_])
        self._check(self._L.sq_score_run_fp8(self._h, _ptr(Hq), _ptr(h_scale), _ptr(Wq), _ptr(w_scale), _ptr(targets), _ptr(cu_seqlens),
                                             T, B, k, window, C.byref(o), self._stream(stream)))
        return out

    def quantize_mx(self, X, operand: int, stream=None, out=None):
        """sq_score_quantize_mx: bf16 [rows, d] -> (uint8 e4m3 codes [rows, d], uint8 scale bytes in the kernel's layout);
        operand = MX_OPERAND_H (token rows) or MX_OPERAND_W (vocabulary rows); `out` = (codes, scales) reuses tensors."""
        import torch
        rows, d = X.shape
        if out is not None:
            q, sf = out
        else:
            q = torch.empty(rows, d, dtype=torch.uint8, device=X.device)
            sf = torch.empty(max(16, self._L.sq_score_mx_scale_bytes(rows, d, operand)), dtype=torch.uint8, device=X.device)
        self._check(self._L.sq_score_quantize_mx(self._h, _ptr(X), rows, operand, _ptr(q), _ptr(sf), self._stream(stream)))
        return q, sf

    def run_mx(self, Hq, h_sf, Wq, w_sf, targets, cu_seqlens, k: int, window: int, stream=None, per_token: bool = True,
               topk: bool = True, out: Optional[dict] = None) -> dict:
        """sq_score_run_mx: the scoring pass on block-scaled (MX) e4m3 operands."""
        T, B = Hq.shape[0], cu_seqlens.shape[0] - 1
        if out is None:
            out = self._alloc_out(T, B, k, Hq.device, per_token, topk)
        o = sq_score_outputs(*[_ptr(out.get(n)) for n, _ in sq_score_outputs._fields_])
        self._check(self._L.sq_score_run_mx(self._h, _ptr(Hq), _ptr(h_sf), _ptr(Wq), _ptr(w_sf), _ptr(targets), _ptr(cu_seqlens),
                                            T, B, k, window, C.byref(o), self._stream(stream)))
        return out

    def run_host(self, H_host, W_dev, targets_host, cu_seqlens_host, k: int, window: int, seq_out_host, stream=None):
        """sq_score_run_host: host inputs -> 4*B host floats (copies are inside the call)."""
        T, B = H_host.shape[0], cu_seqlens_host.shape[0] - 1
        self._check(self._L.sq_score_run_host(self._h, _ptr(H_host), _ptr(W_dev), _ptr(targets_host),
                                              _ptr(cu_seqlens_host), T, B, k, window, _ptr(seq_out_host),
                                              self._stream(stream)))
        return seq_out_host

    def reduce(self, target_logprob, entropy, conf, cu_seqlens, window: int, targets=None, stream=None) -> dict:
        """sq_score_reduce: kernel 2 alone."""
        import torch
        B = cu_seqlens.shape[0] - 1
        out = {n: torch.empty(B, dtype=torch.float32, device=conf.device)
               for n in ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")}
        self._check(self._L.sq_score_reduce(self._h, _ptr(target_logprob), _ptr(entropy), _ptr(conf), _ptr(targets),
                                            _ptr(cu_seqlens), conf.shape[0], B, window,
                                            _ptr(out["seq_mean_logprob"]), _ptr(out["seq_mean_entropy"]),
                                            _ptr(out["seq_mean_conf"]), _ptr(out["seq_min_window_conf"]),
                                            self._stream(stream)))
        return out

    def route(self, seq_conf, group_members, group_offsets, percentile: float, lite_mask=None,
              max_groups_per_problem: Optional[int] = None, stream=None) -> dict:
        """sq_score_route: GC(g), per-problem percentile threshold and routing codes (0 lite / 1 Model 1 / 2 Model 2).
        `group_members` is an int32 [G, K] tensor."""
        import torch
        G, K = group_members.shape
        Q = group_offsets.shape[0] - 1
        dev = seq_conf.device
        if max_groups_per_problem is None:
            off = group_offsets.cpu()
            max_groups_per_problem = int((off[1:] - off[:-1]).max()) if Q > 0 else 0
        out = {"group_fitness": torch.empty(G, dtype=torch.float32, device=dev),
               "theta": torch.empty(Q, dtype=torch.float32, device=dev),
               "route": torch.empty(G, dtype=torch.int32, device=dev)}
        self._check(self._L.sq_score_route(self._h, _ptr(seq_conf), seq_conf.shape[0], _ptr(group_members), _ptr(group_offsets),
                                           Q, G, K, max_groups_per_problem, _ptr(lite_mask), float(percentile),
                                           _ptr(out["group_fitness"]), _ptr(out["theta"]), _ptr(out["route"]),
                                           self._stream(stream)))
        return out

    def select_prob(self, fitness, pop_offsets, zeta: float, stream=None):
        """sq_score_select_prob: softmax(fitness / zeta) within each problem's population."""
        import torch
        prob = torch.empty_like(fitness)
        self._check(self._L.sq_score_select_prob(self._h, _ptr(fitness), _ptr(pop_offsets), pop_offsets.shape[0] - 1,
                                                 float(zeta), _ptr(prob), self._stream(stream)))
        return prob

    def debug_fill_workspace(self, value: int = 0xFF, stream=None):
        """sq_score_debug_fill_workspace (test hook): poison every ctx-owned buffer with a byte pattern."""
        self._check(self._L.sq_score_debug_fill_workspace(self._h, int(value), self._stream(stream)))

    def set_profiling(self, enable: bool):
        self._check(self._L.sq_score_set_profiling(self._h, 1 if enable else 0))

    def kernel_times(self) -> dict:
        """sq_score_kernel_times: ms of the last profiled run's fused / finalize / reduce kernels."""
        ms = (C.c_float * 3)()
        self._check(self._L.sq_score_kernel_times(self._h, ms))
        return {"fused_ms": ms[0], "finalize_ms": ms[1], "reduce_ms": ms[2]}

    def profile_read(self) -> List[dict]:
        """sq_score_profile_read: the same for every profiled run since the last read (at most the newest 64)."""
        ms = (C.c_float * (3 * SQ_PROFILE_RING))()
        n = C.c_int(0)
        self._check(self._L.sq_score_profile_read(self._h, ms, SQ_PROFILE_RING, C.byref(n)))
        return [{"fused_ms": ms[3 * i], "finalize_ms": ms[3 * i + 1], "reduce_ms": ms[3 * i + 2]} for i in range(n.value)]

    def launch_count(self) -> int:
        return self._L.sq_score_launch_count(self._h)

    def last_plan(self) -> Dict[str, int]:
        """sq_score_last_plan: the decomposition the last run launched kernel 1 with (cta_group 4 = quads)."""
        out = sq_score_plan_t()
        rc = self._L.sq_score_last_plan(self._h, C.byref(out))
        if rc != 0:
            raise SqScoreError(rc, "no run with T > 0 on this ctx yet")
        res = {n: getattr(out, n) for n, _ in sq_score_plan_t._fields_ if n != "chunk_vtile"}
        res["chunk_vtile"] = list(out.chunk_vtile[: out.num_chunks + 1])
        return res

    def reduce_form(self) -> str:
        """Form of kernel 2 the last call used (sq_score_reduce_form): 'fused', 'tiles', 'stream', 'tail' or 'none'."""
        return ("none", "fused", "tiles", "stream", "tail")[self._L.sq_score_reduce_form(self._h)]

    def close(self):
        if getattr(self, "_h", None):
            self._L.sq_score_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def shard_sequences(lengths: Sequence[int], world_size: int) -> List[List[int]]:
    """Multi-GPU partition: whole sequences to ranks, longest first onto the
    least-loaded rank (ties -> lowest rank).  No collective on the data path; W is replicated."""
    loads = [0] * world_size
    parts: List[List[int]] = [[] for _ in range(world_size)]
    for i in sorted(range(len(lengths)), key=lambda i: (-int(lengths[i]), i)):
        r = min(range(world_size), key=lambda r: (loads[r], r))
        parts[r].append(i)
        loads[r] += int(lengths[i])
    for p in parts:
        p.sort()
    return parts


def trajectory_positions(query_lens: Sequence[int], traj_lens: Sequence[int]):
    """sq_score_positions_host (host-only, no GPU): for a packed prefill where candidate b is query_lens[b] query
    tokens followed by traj_lens[b] trajectory tokens, returns (pos, cu_seqlens) as int32 lists -- pos[t] is the
    packed row whose hidden state predicts scored token t (the position before it), cu_seqlens
    delimits the trajectories.  Raises ValueError where the library returns INVALID_ARG (a
    trajectory without a query token before it, negative lengths)."""
    B = len(traj_lens)
    if len(query_lens) != B:
        raise ValueError("query_lens and traj_lens differ in length")
    q = (C.c_int32 * max(B, 1))(*[int(v) for v in query_lens])
    n = (C.c_int32 * max(B, 1))(*[int(v) for v in traj_lens])
    cap = sum(max(int(v), 0) for v in traj_lens)
    pos = (C.c_int32 * max(cap, 1))()
    cu = (C.c_int32 * (B + 1))()
    total = C.c_int64(0)
    rc = lib().sq_score_positions_host(q, n, B, pos, cap, cu, C.byref(total))
    if rc != 0:
        raise ValueError("sq_score_positions_host: a trajectory needs at least one query token before it; lengths must be >= 0")
    return list(pos[: total.value]), list(cu)
