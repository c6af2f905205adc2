"""Pins for the CPU oracle (`oracle/sq_oracle.py`): closed forms, invariants, textbook special
cases and pure-Python brute force.  None of these re-types the oracle's own numpy formula: the
brute force below uses only `math` on Python floats, loop by loop, and the closed forms come from
the mathematics (SURVEY.md section 8(c) "What pins each part"; BASELINE.json north_star).

CPU only (`-m "not gpu"`)."""
import math

import numpy as np
import pytest
import torch

from oracle import sq_oracle as O
import workloads


def bf16(x):
    return torch.tensor(x, dtype=torch.float32).to(torch.bfloat16)


# --------------------------------------------------------------------------------------------
# pure-Python brute force of the whole path (independent of numpy/torch arithmetic)
# --------------------------------------------------------------------------------------------
def brute_token(h, W, target, k):
    """h: list[float], W: list[list[float]] -> dict of Python floats.  Eq. 3 by loops."""
    V = len(W)
    z = []
    for v in range(V):
        acc = 0.0
        for j in range(len(h)):
            acc += h[j] * W[v][j]
        z.append(acc)
    m = max(z)
    s = math.fsum(math.exp(zv - m) for zv in z)
    lse = m + math.log(s)
    logp = [zv - lse for zv in z]
    ent = -math.fsum(math.exp(lp) * lp for lp in logp if math.exp(lp) > 0.0)
    order = sorted(range(V), key=lambda v: (-logp[v], v))
    top = order[:k]
    conf = -math.fsum(logp[v] for v in top) / k
    return {"lse": lse, "target_logprob": logp[target], "entropy": ent,
            "topk_index": top, "topk_logprob": [logp[v] for v in top], "conf": conf}


def brute_window_min(c, w):
    L = len(c)
    w = min(w, L)
    best = float("inf")
    for j in range(L - w + 1):
        acc = 0.0
        for i in range(j, j + w):
            acc += c[i]
        best = min(best, acc / w)
    return best


def test_bruteforce_tiny_full_path():
    wl = workloads.custom(d=8, V=37, B=3, len_lo=3, len_hi=9, k=4, window=3, w_std=0.5, seed=11)
    inp = workloads.make_inputs(wl)
    out = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
    Hl = inp["H"].double().tolist()
    Wl = inp["W"].double().tolist()
    tg = inp["targets"].tolist()
    T = inp["T"]
    assert T > 0
    confs, lps, ents = [], [], []
    for t in range(T):
        b = brute_token(Hl[t], Wl, tg[t], wl.k)
        assert out["lse"][t] == pytest.approx(b["lse"], abs=1e-12)
        assert out["target_logprob"][t] == pytest.approx(b["target_logprob"], abs=1e-12)
        assert out["entropy"][t] == pytest.approx(b["entropy"], abs=1e-12)
        assert out["conf"][t] == pytest.approx(b["conf"], abs=1e-12)
        assert list(out["topk_index"][t][:wl.k]) == b["topk_index"]
        np.testing.assert_allclose(out["topk_logprob"][t][:wl.k], b["topk_logprob"], atol=1e-12)
        confs.append(b["conf"]); lps.append(b["target_logprob"]); ents.append(b["entropy"])
    cu = inp["cu_seqlens"].tolist()
    for b in range(inp["B"]):
        lo, hi = cu[b], cu[b + 1]
        L = hi - lo
        assert out["seq_mean_logprob"][b] == pytest.approx(sum(lps[lo:hi]) / L, abs=1e-12)
        assert out["seq_mean_entropy"][b] == pytest.approx(sum(ents[lo:hi]) / L, abs=1e-12)
        assert out["seq_mean_conf"][b] == pytest.approx(sum(confs[lo:hi]) / L, abs=1e-12)
        assert out["seq_min_window_conf"][b] == pytest.approx(brute_window_min(confs[lo:hi], wl.window), abs=1e-12)


# --------------------------------------------------------------------------------------------
# a1 logits
# --------------------------------------------------------------------------------------------
def test_logits_d1_and_operand_order():
    # d = 1: z[t,v] = h[t] * w[v]; non-square so a transposed operand cannot pass.
    H = bf16([[2.0], [-3.0], [0.5]])
    W = bf16([[1.0], [4.0], [-0.25], [8.0], [0.0]])
    z = O.logits(H, O.widen(W))
    assert z.shape == (3, 5)
    expect = [[2, 8, -0.5, 16, 0], [-3, -12, 0.75, -24, 0], [0.5, 2, -0.125, 4, 0]]
    assert z.tolist() == expect


def test_logits_exact_integers():
    # small-integer bf16 values: every partial sum is an exact integer
    rng = np.random.default_rng(3)
    Hn = rng.integers(-4, 5, size=(5, 7)); Wn = rng.integers(-4, 5, size=(6, 7))
    z = O.logits(bf16(Hn.tolist()), O.widen(bf16(Wn.tolist())))
    for t in range(5):
        for v in range(6):
            assert z[t, v] == sum(int(Hn[t, j]) * int(Wn[v, j]) for j in range(7))


def test_bf16_widening_is_exact():
    x = torch.randn(1000, generator=torch.Generator().manual_seed(0)).to(torch.bfloat16)
    assert torch.equal(O.widen(x).to(torch.bfloat16), x)
    assert torch.equal(O.widen(x).float(), x.float())


# --------------------------------------------------------------------------------------------
# identical W rows: the BASELINE.json pins
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("V", [1, 2, 7, 1000])
def test_identical_rows(V):
    g = torch.Generator().manual_seed(5)
    d = 16
    w = (torch.randn(d, generator=g) * 0.3).to(torch.bfloat16)
    W = w.repeat(V, 1)
    H = torch.randn(6, d, generator=g).to(torch.bfloat16)
    k = min(3, V)
    r = O.token_scores(H, O.widen(W), [0, V - 1, V // 2, 0, 0, 0], k)
    zrow = (H.double() @ w.double()).numpy()
    lnV = math.log(V)
    np.testing.assert_allclose(r["lse"], zrow + lnV, atol=1e-12)
    np.testing.assert_allclose(r["target_logprob"], -lnV, atol=1e-12)
    np.testing.assert_allclose(r["entropy"], lnV, atol=1e-12)
    np.testing.assert_allclose(r["topk_logprob"], -lnV, atol=1e-12)
    np.testing.assert_allclose(r["conf"], lnV, atol=1e-12)
    # ties -> ascending index
    assert r["topk_index"][0].tolist() == list(range(min(V, k + 1)))


# --------------------------------------------------------------------------------------------
# V = 2 textbook forms: softplus / binary entropy
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("delta", [0.0, 0.5, -2.0, 8.0, -40.0])
def test_two_class_closed_forms(delta):
    # h = [1, 0]; W = [[a, *], [b, *]] -> z = (a, b), delta = a - b (all bf16-exact values)
    a, b = (delta, 0.0)
    H = bf16([[1.0, 0.0]])
    W = bf16([[a, 3.0], [b, -1.0]])
    r = O.token_scores(H, O.widen(W), [0], 1)
    softplus = lambda x: max(x, 0.0) + math.log1p(math.exp(-abs(x)))
    assert r["lse"][0] == pytest.approx(max(a, b) + math.log1p(math.exp(-abs(delta))), abs=1e-13)
    assert r["target_logprob"][0] == pytest.approx(-softplus(b - a), abs=1e-13)
    p = 1.0 / (1.0 + math.exp(-delta))
    hb = 0.0
    for q in (p, 1.0 - p):
        if q > 0.0:
            hb -= q * math.log(q)
    assert r["entropy"][0] == pytest.approx(hb, abs=1e-13)
    # k = 1: the top log-prob is -log s = max - lse
    assert r["topk_logprob"][0][0] == pytest.approx(max(a, b) - r["lse"][0], abs=1e-13)
    assert r["topk_index"][0][0] == (0 if a >= b else 1)


# --------------------------------------------------------------------------------------------
# one hot + flat rest: closed-form softmax statistics
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("alpha,V", [(3.0, 50), (16.0, 1000), (0.0, 9), (-2.0, 33)])
def test_onehot_plus_flat(alpha, V):
    d = 4
    H = bf16([[1.0, 0.0, 0.0, 0.0]])
    Wm = torch.zeros(V, d)
    hot = V // 3
    Wm[hot, 0] = alpha
    Wm[:, 1:] = 0.75          # columns that h does not see
    r = O.token_scores(H, O.widen(Wm.to(torch.bfloat16)), [hot], 2)
    denom = math.exp(alpha) + (V - 1)
    p1 = math.exp(alpha) / denom
    rest = (1.0 - p1)
    ent = -p1 * math.log(p1) - (rest * math.log(rest / (V - 1)) if rest > 0 else 0.0)
    assert r["lse"][0] == pytest.approx(math.log(denom), abs=1e-12)
    assert r["target_logprob"][0] == pytest.approx(alpha - math.log(denom), abs=1e-12)
    assert r["entropy"][0] == pytest.approx(ent, abs=1e-12)
    if alpha > 0:
        assert r["topk_index"][0][0] == hot
        # Eq. 3 with k = 2: mean of the hot log-prob and one flat log-prob, negated
        assert r["conf"][0] == pytest.approx(-0.5 * ((alpha - math.log(denom)) + (0.0 - math.log(denom))), abs=1e-12)


# --------------------------------------------------------------------------------------------
# invariants on random inputs
# --------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def tiny_scored():
    inp = workloads.make_inputs(workloads.CONFIGS["tiny"])
    out = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], inp["k"], inp["window"])
    return inp, out


def test_tiny_config_shape(tiny_scored):
    inp, out = tiny_scored
    assert inp["T"] == 256 and inp["B"] == 4 and inp["W"].shape == (1024, 64)
    L = np.diff(inp["cu_seqlens"].numpy())
    assert L.min() >= 32 and L.max() <= 96
    assert out["topk_logprob"].shape == (256, 6)


def test_probabilities_sum_to_one_and_bounds(tiny_scored):
    inp, out = tiny_scored
    r = O.token_scores(inp["H"][:32], O.widen(inp["W"]), inp["targets"][:32].numpy(), inp["k"])
    np.testing.assert_allclose(np.exp(r["logp"]).sum(axis=1), 1.0, atol=1e-12)
    V, k = 1024, inp["k"]
    assert (out["entropy"] >= 0).all() and (out["entropy"] <= math.log(V) + 1e-12).all()
    assert (out["target_logprob"] <= 0).all()
    assert (out["topk_logprob"][:, 0] >= -math.log(V) - 1e-12).all()
    assert (np.diff(out["topk_logprob"], axis=1) <= 0).all()         # non-increasing
    assert (out["conf"] >= math.log(k) - 1e-12).all()                # Jensen (reading #2)
    # the target's log-prob can never exceed the top-1 log-prob
    assert (out["target_logprob"] <= out["topk_logprob"][:, 0] + 1e-15).all()


def test_k_equals_V_gives_all_logprobs():
    wl = workloads.custom(d=8, V=12, B=1, len_lo=4, len_hi=4, k=12, seed=3, w_std=1.0)
    inp = workloads.make_inputs(wl)
    r = O.token_scores(inp["H"], O.widen(inp["W"]), inp["targets"].numpy(), 12)
    assert r["topk_logprob"].shape == (4, 12)
    np.testing.assert_allclose(np.exp(r["topk_logprob"]).sum(axis=1), 1.0, atol=1e-12)
    for t in range(4):
        assert sorted(r["topk_index"][t].tolist()) == list(range(12))


def test_logit_shift_invariance():
    # a constant W column c seen by H[:,col] = a shifts every logit by a*c: lse shifts, the rest does not.
    wl = workloads.custom(d=8, V=64, B=1, len_lo=5, len_hi=5, k=3, seed=9, w_std=0.5)
    inp = workloads.make_inputs(wl)
    H0 = inp["H"].clone(); W0 = inp["W"].clone()
    H0[:, 7] = 0.0
    base = O.token_scores(H0, O.widen(W0), inp["targets"].numpy(), 3)
    for a, c in [(8.0, 10.0), (-8.0, 10.0)]:
        H1 = H0.clone(); W1 = W0.clone()
        H1[:, 7] = a; W1[:, 7] = c
        r = O.token_scores(H1, O.widen(W1), inp["targets"].numpy(), 3)
        np.testing.assert_allclose(r["lse"], base["lse"] + a * c, atol=1e-10)
        for key in ("target_logprob", "entropy", "conf", "topk_logprob"):
            np.testing.assert_allclose(r[key], base[key], atol=1e-10)
        assert (r["topk_index"] == base["topk_index"]).all()


def test_vocab_permutation_invariance():
    wl = workloads.custom(d=8, V=300, B=1, len_lo=6, len_hi=6, k=5, seed=13, w_std=0.7)
    inp = workloads.make_inputs(wl)
    base = O.token_scores(inp["H"], O.widen(inp["W"]), inp["targets"].numpy(), 5)
    perm = torch.randperm(300, generator=torch.Generator().manual_seed(1))
    Wp = inp["W"][perm]                     # new row i = old row perm[i]
    inv = torch.empty_like(perm); inv[perm] = torch.arange(300)
    r = O.token_scores(inp["H"], O.widen(Wp), inv[inp["targets"].long()].numpy(), 5)
    for key in ("lse", "target_logprob", "entropy", "conf", "topk_logprob"):
        np.testing.assert_allclose(r[key], base[key], atol=1e-12)
    assert (perm.numpy()[r["topk_index"]] == base["topk_index"]).all()


def test_topk_planted_maximum_positions():
    V, d = 600, 4
    for col in (0, 127, 128, 255, 256, V - 1):
        Wm = torch.zeros(V, d); Wm[col, 0] = 5.0; Wm[(col + 7) % V, 0] = 2.0
        r = O.token_scores(bf16([[1.0, 0, 0, 0]]), O.widen(Wm.to(torch.bfloat16)), [col], 2)
        assert r["topk_index"][0][:2].tolist() == [col, (col + 7) % V]
        assert r["target_logprob"][0] == r["topk_logprob"][0][0]


def test_no_target_extension():
    wl = workloads.custom(d=8, V=20, B=1, len_lo=4, len_hi=4, k=2, seed=4)
    inp = workloads.make_inputs(wl)
    tg = inp["targets"].numpy().copy(); tg[1] = -1; tg[2] = 20
    out = O.score(inp["H"], inp["W"], tg, inp["cu_seqlens"], 2, 3)
    assert out["target_logprob"][1] == 0.0 and out["target_logprob"][2] == 0.0
    assert out["seq_mean_logprob"][0] == pytest.approx((out["target_logprob"][0] + out["target_logprob"][3]) / 2)


def test_peaked_rows_have_larger_conf():
    # peaked distribution -> c(i) large, flat -> small.  (Strong peak: p_top -> 1 pushes
    # every other log-prob far down.  A *mild* peak lowers c(i) instead -- see DESIGN.md reading #2.)
    wl = workloads.custom(d=64, V=512, B=1, len_lo=64, len_hi=64, k=5, seed=21, w_std=0.05,
                          planted_frac=0.5, planted_scale=400.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    out = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], 5, 8)
    pl = inp["planted"].numpy()
    assert pl.any() and (~pl).any()
    assert out["conf"][pl].mean() > out["conf"][~pl].mean()
    assert out["entropy"][pl].mean() < out["entropy"][~pl].mean()


def test_matches_torch_library_routines(tiny_scored):
    # library cross-check (extra, not the pin): logsumexp / log_softmax / topk in fp64
    inp, out = tiny_scored
    z = inp["H"].double() @ inp["W"].double().T
    np.testing.assert_allclose(out["lse"], torch.logsumexp(z, 1).numpy(), atol=1e-12)
    lsm = torch.log_softmax(z, 1)
    tv, _ = torch.topk(lsm, 5, dim=1)
    np.testing.assert_allclose(out["topk_logprob"][:, :5], tv.numpy(), atol=1e-12)
    ent = -(lsm.exp() * lsm).sum(1)
    np.testing.assert_allclose(out["entropy"], ent.numpy(), atol=1e-12)


# --------------------------------------------------------------------------------------------
# a7 per-sequence reductions
# --------------------------------------------------------------------------------------------
def test_window_min_special_cases():
    rng = np.random.default_rng(0)
    c = rng.uniform(2.0, 9.0, size=37)
    assert O.window_min_mean(c, 1) == c.min()                                  # w = 1 -> min
    assert O.window_min_mean(c, 37) == pytest.approx(c.mean(), abs=1e-14)      # w = L -> mean
    assert O.window_min_mean(c, 1000) == pytest.approx(c.mean(), abs=1e-14)    # w > L -> mean
    assert O.window_min_mean(np.full(20, 4.25), 7) == 4.25                     # constant
    assert math.isnan(O.window_min_mean(np.zeros(0), 4))                       # L = 0
    for w in (2, 5, 16):
        assert O.window_min_mean(c, w) == pytest.approx(brute_window_min(c.tolist(), w), abs=1e-13)
        assert O.window_min_mean(c, w) >= c.min()


def test_window_min_step_function():
    # conf = 10 for 6 tokens, then 2 for 3 tokens, then 10 for 6: w=4 -> best window holds 3 twos and one ten
    c = np.array([10.0] * 6 + [2.0] * 3 + [10.0] * 6)
    assert O.window_min_mean(c, 4) == (3 * 2.0 + 10.0) / 4
    assert O.window_min_mean(c, 3) == 2.0
    assert O.window_min_mean(c, 2) == 2.0
    assert O.window_min_mean(c, 15) == pytest.approx((12 * 10 + 6) / 15)


def test_window_min_below_sequence_mean():
    # the mean of all window means with equal weight need not equal the sequence mean, but the
    # minimum window mean is <= the sequence mean whenever w divides L (windows tile the sequence)
    rng = np.random.default_rng(4)
    c = rng.uniform(0, 5, size=48)
    for w in (1, 2, 3, 4, 6, 8, 12, 16, 24, 48):
        assert O.window_min_mean(c, w) <= c.mean() + 1e-12


def test_sequence_scores_segments_and_empty():
    lp = -np.arange(1, 11, dtype=np.float64)
    en = np.arange(10, dtype=np.float64) * 0.5
    cf = np.array([3, 1, 4, 1, 5, 9, 2, 6, 5, 3], dtype=np.float64)
    cu = [0, 4, 4, 5, 10]                       # lengths 4, 0, 1, 5
    s = O.sequence_scores(lp, en, cf, cu, window=2)
    assert s["seq_mean_logprob"][0] == -2.5 and s["seq_mean_entropy"][0] == 0.75
    assert s["seq_mean_conf"][0] == 2.25 and s["seq_min_window_conf"][0] == 2.0
    assert all(math.isnan(s[key][1]) for key in s)
    assert s["seq_mean_conf"][2] == 5.0 and s["seq_min_window_conf"][2] == 5.0      # L = 1 < w
    assert s["seq_mean_logprob"][3] == -8.0
    assert s["seq_min_window_conf"][3] == 4.0                                        # (5+3)/2
    assert s["seq_mean_conf"][3] == 5.0


def test_per_token_outputs_do_not_depend_on_cu_seqlens(tiny_scored):
    inp, out = tiny_scored
    out2 = O.score(inp["H"], inp["W"], inp["targets"], torch.tensor([0, 256]), inp["k"], inp["window"])
    for key in ("lse", "target_logprob", "entropy", "conf"):
        assert (out[key] == out2[key]).all()
    assert out2["seq_mean_conf"][0] == pytest.approx(out["conf"].mean(), abs=1e-13)


# --------------------------------------------------------------------------------------------
# golden fixture (written by tests/golden/make_golden.py, which calls only oracle/)
# --------------------------------------------------------------------------------------------
def test_golden_fixture_regression(tiny_scored):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "tiny_sequence_scores.txt")
    inp, out = tiny_scored
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 4
    for b, row in enumerate(rows):
        vals = [float(x) for x in row[2:]]
        assert int(row[1]) == int(inp["cu_seqlens"][b + 1] - inp["cu_seqlens"][b])
        got = [out[key][b] for key in ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")]
        np.testing.assert_allclose(got, vals, rtol=0, atol=1e-11)
