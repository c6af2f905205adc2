"""CPU fp64 ORACLE for the sq_score hot path.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this file.  It shares no code with `paper_2604_07725_b200/` (the CUDA path) and
never imports it.  It is deliberately plain and slow: every function is the *definition* of the
quantity written out in fp64 (numpy / torch CPU ops), in the paper's notation, with no blocking,
fusion, online update or reordering, so it can be checked against the paper by eye.

What the path computes:

  z[t,v]   = sum_j H[t,j] * W[v,j]                       LM-head logits (prefill-only scoring pass,
                                                          PAPER.md:163, 199-203); bf16 inputs are widened
                                                          to fp64 exactly, bf16*bf16 products are exact.
  log p    = z - logsumexp_v z                           softmax at temperature 1, no bias (reading #5)
  target_logprob[t] = log p[t, targets[t]]               "cross-model log-probabilities", PAPER.md:84
  entropy[t]        = - sum_v p log p   (nats)           BASELINE.json north_star (not in the paper)
  top-K_l log-probs, descending, ties by ascending index PAPER.md:149-158
  conf[t] = c(i) = -(1/K_l) * sum_{j<=K_l} log p(v_j)    Eq. 3
  C(tau)  = (1/|tau|) * sum_i c(i)                       Eq. 4 (left)
  per-sequence mean target_logprob / mean entropy        BASELINE.json north_star
  min over stride-1 full windows of length w'=min(w,L) of the window mean of c(i)
                                                          BASELINE.json north_star (readings #9, #10)

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): every function below is pinned to closed forms,
invariants or pure-Python brute force -- see the table in DESIGN.md "Oracle and its pins".
No function here is "parity unpinned".
"""
from __future__ import annotations

import math

import numpy as np
import torch

ORACLE_VERSION = 5


def widen(x_bf16: torch.Tensor) -> torch.Tensor:
    """bf16 -> fp64 (exact)."""
    return x_bf16.to(torch.float64)


def logits(H_rows: torch.Tensor, W64: torch.Tensor) -> np.ndarray:
    """z[t,v] = sum_j H[t,j] * W[v,j] in fp64.  The library matmul is the step (a dgemm); its
    summation order is irrelevant at the 1e-16 level because every product is exact in fp64."""
    return (widen(H_rows) @ W64.T).numpy()


def token_scores(H_rows: torch.Tensor, W64: torch.Tensor, targets_rows, k: int, extra: int = 1) -> dict:
    """Per-token outputs for the given rows.  `W64 = widen(W)` is passed in so that callers can
    convert the LM head once.  Returns k+extra top entries (the extra one lets the parity checker
    see the gap below the k-th entry, reading #7); `conf` uses exactly the first k (Eq. 3)."""
    z = logits(H_rows, W64)                                   # [n, V]
    n, V = z.shape
    tg = np.asarray(targets_rows, dtype=np.int64)
    m = z.max(axis=1)                                         # two-pass logsumexp (not online)
    s = np.exp(z - m[:, None]).sum(axis=1)
    lse = m + np.log(s)
    logp = z - lse[:, None]                                   # log p_theta(v | t_<i, Q)
    valid = (tg >= 0) & (tg < V)                              # targets outside [0,V) = "no target"
    target_logprob = np.where(valid, logp[np.arange(n), np.where(valid, tg, 0)], 0.0)
    p = np.exp(logp)
    plogp = np.where(p > 0.0, p * logp, 0.0)                  # 0 * log 0 := 0
    entropy = -plogp.sum(axis=1)
    kk = min(V, k + extra)
    order = np.argsort(-logp, axis=1, kind="stable")[:, :kk]  # value desc, index asc on ties
    topk_logprob = np.take_along_axis(logp, order, axis=1)
    conf = -topk_logprob[:, :k].sum(axis=1) / k               # Eq. 3
    return {"lse": lse, "target_logprob": target_logprob, "target_valid": valid, "entropy": entropy,
            "topk_logprob": topk_logprob, "topk_index": order.astype(np.int64), "conf": conf,
            "logp": logp}


def window_min_mean(conf_seq: np.ndarray, window: int) -> float:
    """min_j (1/w') * sum_{i=j}^{j+w'-1} conf[i], w' = min(window, L), j = 0..L-w' (stride 1, full
    windows only; reading #9).  Direct re-summation of every window -- no prefix sums."""
    L = len(conf_seq)
    if L == 0:
        return float("nan")
    w = min(int(window), L)
    best = np.inf
    for j in range(0, L - w + 1):
        best = min(best, float(np.sum(conf_seq[j:j + w], dtype=np.float64)) / w)
    return best


def sequence_scores(target_logprob, entropy, conf, cu_seqlens, window: int, target_valid=None) -> dict:
    """Per-sequence varlen reductions over tokens [cu[b], cu[b+1]).  Means are arithmetic means
    over the L tokens (Eq. 4 left for conf); the mean target log-prob counts only valid targets
    (reading #11).  Empty sequences (and sequences with no valid target, for the log-prob mean)
    give NaN."""
    lp = np.asarray(target_logprob, dtype=np.float64)
    en = np.asarray(entropy, dtype=np.float64)
    cf = np.asarray(conf, dtype=np.float64)
    cu = np.asarray(cu_seqlens, dtype=np.int64)
    ok = np.ones(len(lp), dtype=bool) if target_valid is None else np.asarray(target_valid, dtype=bool)
    B = len(cu) - 1
    out = {key: np.full(B, np.nan) for key in
           ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")}
    for b in range(B):
        lo, hi = int(cu[b]), int(cu[b + 1])
        L = hi - lo
        if L <= 0:
            continue
        nvalid = int(ok[lo:hi].sum())
        if nvalid > 0:
            out["seq_mean_logprob"][b] = float(np.sum(lp[lo:hi][ok[lo:hi]])) / nvalid
        out["seq_mean_entropy"][b] = float(np.sum(en[lo:hi])) / L
        out["seq_mean_conf"][b] = float(np.sum(cf[lo:hi])) / L          # C(tau), Eq. 4
        out["seq_min_window_conf"][b] = window_min_mean(cf[lo:hi], window)
    return out


def score(H: torch.Tensor, W: torch.Tensor, targets, cu_seqlens, k: int, window: int,
          row_batch: int = 64) -> dict:
    """Whole path on all rows (small cases): per-token scores, then per-sequence reductions."""
    W64 = widen(W)
    T = H.shape[0]
    tg = np.asarray(targets, dtype=np.int64)
    keys = ("lse", "target_logprob", "target_valid", "entropy", "topk_logprob", "topk_index", "conf", "logp")
    parts = {key: [] for key in keys}
    for r0 in range(0, T, row_batch):
        r = token_scores(H[r0:r0 + row_batch], W64, tg[r0:r0 + row_batch], k)
        for key in keys:
            parts[key].append(r[key])
    V = W.shape[0]
    kk = min(V, k + 1)
    tok = {key: (np.concatenate(parts[key]) if T > 0 else
                 np.zeros((0, kk) if key.startswith("topk") else ((0, V) if key == "logp" else (0,))))
           for key in keys}
    seq = sequence_scores(tok["target_logprob"], tok["entropy"], tok["conf"], cu_seqlens, window,
                          tok["target_valid"])
    tok.update(seq)
    return tok


# ------------------------------------------------------------------------------------------------
# Next row: group fitness, per-problem percentile threshold, routing,
# fitness-weighted selection probabilities
# ------------------------------------------------------------------------------------------------
def group_confidence(seq_conf, group_members) -> np.ndarray:
    """GC(g) = (1/K) * sum_{tau in g} C(tau) -- Eq. 4 (right).  `group_members` is
    [G, K] indices into seq_conf; K = |g| (reading #12)."""
    c = np.asarray(seq_conf, dtype=np.float64)
    gm = np.asarray(group_members, dtype=np.int64)
    return c[gm].sum(axis=1) / gm.shape[1]


def percentile_threshold(values, p: float) -> float:
    """theta = Percentile_p(values) -- Eq. 6.  The paper does not say how to
    interpolate; reading #13: linear interpolation between order statistics at rank p/100*(n-1)
    (NumPy's default).  Empty input -> NaN."""
    v = np.sort(np.asarray(values, dtype=np.float64))
    n = len(v)
    if n == 0:
        return float("nan")
    pos = (p / 100.0) * (n - 1)
    lo = int(math.floor(pos))
    hi = min(lo + 1, n - 1)
    return float(v[lo] + (pos - lo) * (v[hi] - v[lo]))


def route(seq_conf, group_members, group_offsets, p: float, lite_mask=None) -> dict:
    """Per problem q (groups [off[q], off[q+1])): F(g) = GC(g); theta_q over the non-lite groups
    (Eq. 6); mu(g,q) = Model 1 if GC(g) > theta_q ("easy", strict) else Model 2 (Eq. 7).
    Codes: 0 = B_lite (given by `lite_mask`; the consensus test itself is on answer strings and is
    out of scope), 1 = Model 1, 2 = Model 2, 3 = fitness undefined: a group whose GC is not finite
    (it holds an empty trajectory, whose C(tau) is NaN) takes no part in the percentile and is left
    to the caller (reading #24; the paper never scores an empty trajectory)."""
    gc = group_confidence(seq_conf, group_members)
    off = np.asarray(group_offsets, dtype=np.int64)
    G = len(gc)
    lite = np.zeros(G, dtype=bool) if lite_mask is None else np.asarray(lite_mask, dtype=bool)
    theta = np.full(len(off) - 1, np.nan)
    code = np.zeros(G, dtype=np.int32)
    for q in range(len(off) - 1):
        idx = np.arange(off[q], off[q + 1])
        undefined = idx[~lite[idx] & ~np.isfinite(gc[idx])]
        code[undefined] = 3
        live = idx[~lite[idx] & np.isfinite(gc[idx])]
        theta[q] = percentile_threshold(gc[live], p)
        for g in live:
            code[g] = 1 if gc[g] > theta[q] else 2
    return {"group_fitness": gc, "theta": theta, "route": code}


def selection_probabilities(fitness, pop_offsets, zeta: float) -> np.ndarray:
    """Fitness-weighted selection: candidate i of problem q is drawn with probability
    exp(f_i / zeta) / sum_j exp(f_j / zeta) over the problem's population."""
    fv = np.asarray(fitness, dtype=np.float64)
    off = np.asarray(pop_offsets, dtype=np.int64)
    out = np.zeros_like(fv)
    for q in range(len(off) - 1):
        x = fv[off[q]:off[q + 1]] / zeta
        if len(x):
            e = np.exp(x - x.max())
            out[off[q]:off[q + 1]] = e / e.sum()
    return out


# ------------------------------------------------------------------------------------------------
# Next row: the step before the path -- gather the positions whose next-token
# distribution is wanted and apply the scorer's final RMSNorm, giving the H the scoring pass consumes
# ------------------------------------------------------------------------------------------------
def trajectory_positions(query_lens, traj_lens):
    """Packed prefill of B candidates, candidate b occupying query_lens[b] query tokens followed by
    traj_lens[b] trajectory tokens.  Token i of the trajectory (i = 1..|tau|) is scored by
    log p(. | t_<i, Q) (Eq. 3), i.e. by the hidden state of the position just before
    it (reading #3); only the |tau| trajectory tokens are averaged (Eq. 4; reading #4).
    Returns (pos, cu_seqlens): pos[t] = row of the packed hidden states that predicts scored token t.
    A candidate with an empty query has no state that predicts its first token: ValueError."""
    pos, cu, base = [], [0], 0
    for q, L in zip(query_lens, traj_lens):
        q, L = int(q), int(L)
        if q < 1 and L > 0:
            raise ValueError("a trajectory needs at least one query token before it")
        first = base + q               # packed index of trajectory token 1
        for i in range(L):
            pos.append(first + i - 1)  # the state of the previous position predicts token i
        cu.append(cu[-1] + L)
        base += q + L
    return np.asarray(pos, dtype=np.int64), np.asarray(cu, dtype=np.int64)


def prepare_hidden(X: torch.Tensor, pos, gain: torch.Tensor, eps: float) -> np.ndarray:
    """h[t,:] = x / sqrt(mean_j x_j^2 + eps) * gain with x = X[pos[t],:] -- the RMSNorm that closes the
    model families whose (d, V) the configs borrow; the paper does not describe the scorer's
    internals (reading #20: all arithmetic before ONE rounding to bf16).  fp64 throughout;
    returns the unrounded fp64 rows [T, d]."""
    x = widen(X)[torch.as_tensor(np.asarray(pos, dtype=np.int64))].numpy()
    g = widen(gain).numpy()
    ms = (x * x).sum(axis=1) / x.shape[1]
    return x / np.sqrt(ms + eps)[:, None] * g[None, :]


def round_to_bf16(h64: np.ndarray) -> torch.Tensor:
    """Nearest-even rounding fp64 -> bf16 (one rounding; torch's conversion is the library step)."""
    return torch.from_numpy(np.ascontiguousarray(h64)).to(torch.bfloat16)


def bf16_half_ulp(h64: np.ndarray) -> np.ndarray:
    """Half a bf16 unit in the last place at |h| (8 significand bits; subnormals below 2^-126)."""
    a = np.abs(h64)
    e = np.floor(np.log2(np.maximum(a, 2.0 ** -126)))
    return 0.5 * 2.0 ** (e - 7)


# ------------------------------------------------------------------------------------------------
# Next row (SURVEY section 8(f)-4, FP8 variant): e4m3 quantisation with per-row / per-tensor scales,
# by its definition in fp64: scale = amax / 448, code = the e4m3 value nearest to x / scale (ties to the
# even mantissa).  The codes are a quantised representation decided by floating point; the CUDA path
# takes that decision in fp32, so the parity test accepts a code that is a correct rounding of a value
# within a stated fp32 slack of x / scale and demands the code below except within that slack of a
# rounding boundary (reading #23).  Everything after it (the scoring of the dequantised
# operands) is the fp64 path above.
# ------------------------------------------------------------------------------------------------
E4M3_MAX = 448.0


def e4m3_values() -> np.ndarray:
    """The 256 e4m3 ("fn": no infinities, S.1111.111 = NaN) code points as fp64, by their definition:
    sign, 4 exponent bits (bias 7), 3 mantissa bits; exponent 0 = subnormal (mantissa / 8 * 2^-6)."""
    vals = np.empty(256)
    for c in range(256):
        sgn = -1.0 if c & 0x80 else 1.0
        e, m = (c >> 3) & 0xF, c & 0x7
        if e == 0xF and m == 0x7:
            vals[c] = np.nan
        elif e == 0:
            vals[c] = sgn * (m / 8.0) * 2.0 ** -6
        else:
            vals[c] = sgn * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return vals


def round_to_e4m3(y: np.ndarray) -> np.ndarray:
    """Codes of the e4m3 values nearest to y (|y| <= 448), ties to the even mantissa.  Written as a search
    over the 127 non-negative code points -- the definition of rounding to nearest -- not a bit trick."""
    pos = e4m3_values()[:127]                     # codes 0 .. 126 = 0 .. 448 ascending
    a = np.abs(np.asarray(y, dtype=np.float64))
    hi = np.searchsorted(pos, a, side="left").clip(1, 126)
    lo = hi - 1
    dlo, dhi = a - pos[lo], pos[hi] - a
    pick_hi = (dhi < dlo) | ((dhi == dlo) & (hi % 2 == 0))   # even code = even mantissa
    code = np.where(pick_hi, hi, lo).astype(np.uint8)
    code = np.where(a == 0, 0, code).astype(np.uint8)
    return np.where(np.signbit(y), code | 0x80, code).astype(np.uint8)


def quantize_fp8(X: torch.Tensor, per_tensor: bool):
    """(codes uint8 [rows, d], scales fp64 [rows] or [1], y fp64 [rows, d]) with scale = amax / 448 (1 where
    amax = 0), y = x / scale the exact scaled values and codes = round_to_e4m3(y), so that
    x ~= e4m3_values()[code] * scale.  amax is taken per row, or over the whole tensor."""
    x = widen(X).numpy()
    amax = np.abs(x).max() if per_tensor else np.abs(x).max(axis=1)
    amax = np.asarray(amax, dtype=np.float64).reshape(-1)
    scale = np.where(amax > 0, amax / E4M3_MAX, 1.0)
    y = x / (scale[0] if per_tensor else scale[:, None])
    return round_to_e4m3(y), scale, y


def e4m3_half_ulp(y: np.ndarray) -> np.ndarray:
    """Half the spacing of the e4m3 code points around |y| <= 448: 3 mantissa bits, spacing 2^(e-3) in the
    binade [2^e, 2^(e+1)), e >= -6; below the first normal (2^-6) the subnormal spacing 2^-9."""
    a = np.abs(np.asarray(y, dtype=np.float64))
    e = np.floor(np.log2(np.maximum(a, 2.0 ** -6)))
    return 0.5 * 2.0 ** (np.minimum(e, 8.0) - 3)


def dequantize_fp8(codes: np.ndarray, scale: np.ndarray) -> torch.Tensor:
    """fp64 tensor codes * scale (exact: an e4m3 value times an fp32 scale fits fp64)."""
    v = e4m3_values()[codes]
    s = np.asarray(scale, dtype=np.float64)
    return torch.from_numpy(v * (s[0] if s.size == 1 else s[:, None]))


# ------------------------------------------------------------------------------------------------
# Next widening (block-scaled variant): MX-style e4m3 with one power-of-two scale per
# block of 32 consecutive elements of a row (the format tcgen05.mma.kind::mxf8f6f4.block_scale consumes:
# e4m3 elements, UE8M0 scales = 2^(code - 127)).  By definition, in exact arithmetic (reading #26):
#   e_blk  = the smallest integer e with amax_blk <= 448 * 2^e   (no element saturates; amax = 0: e = -127)
#   code   = the e4m3 value nearest to x / 2^e_blk (ties to the even mantissa)
#   x     ~= e4m3_values()[code] * 2^e_blk
# Scaling by a power of two is exact, so the CUDA path must reproduce codes and exponents bit for bit.
# ------------------------------------------------------------------------------------------------
MX_BLOCK = 32


def quantize_mx(X: torch.Tensor):
    """(codes uint8 [rows, d], exps int32 [rows, ceil(d / 32)]) -- see the definition above.  A ragged last block
    (d % 32 != 0) is scaled by the maximum of the elements it has."""
    x = widen(X).numpy()
    rows, d = x.shape
    nb = -(-d // MX_BLOCK)
    xp = np.zeros((rows, nb * MX_BLOCK))
    xp[:, :d] = x
    blk = xp.reshape(rows, nb, MX_BLOCK)
    amax = np.abs(blk).max(axis=2)
    m, ex = np.frexp(amax / E4M3_MAX)              # amax / 448 = m * 2^ex, m in [0.5, 1): exact (a division by 7 * 2^6 ...
    # ... is not exact in general, so decide by the exact comparison amax <= 448 * 2^e instead of trusting m)
    e = ex.astype(np.int64)                        # candidate: 2^ex > amax / 448 always holds (m < 1)
    ok_lower = amax <= E4M3_MAX * np.exp2((e - 1).astype(np.float64))   # 448 * 2^(e-1) is exact in fp64
    e = np.where(ok_lower, e - 1, e)
    e = np.where(amax > 0, np.clip(e, -127, 127), -127).astype(np.int32)
    y = blk / np.exp2(e.astype(np.float64))[:, :, None]
    codes = round_to_e4m3(y).reshape(rows, nb * MX_BLOCK)[:, :d]
    return np.ascontiguousarray(codes), e


def dequantize_mx(codes: np.ndarray, exps: np.ndarray) -> torch.Tensor:
    """fp64 tensor e4m3_values()[code] * 2^exp of the element's block (exact)."""
    v = e4m3_values()[codes]
    rows, d = v.shape
    s = np.repeat(np.exp2(exps.astype(np.float64)), MX_BLOCK, axis=1)[:, :d]
    return torch.from_numpy(v * s)
