"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element on
the same seeded inputs.  Tolerances are BASELINE.json north_star's:
  abs 2e-3 on logsumexp, target log-prob and top-k values (and conf, their mean);
  rel 1e-3 on entropy and the sequence aggregates;
  top-k indices exact wherever adjacent oracle values differ by more than 1e-2.
"""
import math

import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O

pytestmark = pytest.mark.gpu

ABS_TOL = 2e-3
REL_TOL = 1e-3
GAP = 1e-2
SEQ_KEYS = ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")


def _sq():
    import paper_2604_07725_b200 as sq
    return sq


def run_gpu(inp, k=None, window=None, targets=None, **eng_kw):
    sq = _sq()
    wl = inp["workload"]
    k = wl.k if k is None else k
    window = wl.window if window is None else window
    dev = torch.device("cuda:0")
    eng = sq.SqScore(wl.d, wl.V, max_tokens=max(1, inp["T"]), max_seqs=max(1, inp["B"]), max_k=k, **eng_kw)
    tg = inp["targets"] if targets is None else targets
    out = eng.run(inp["H"].to(dev), inp["W"].to(dev), tg.to(dev), inp["cu_seqlens"].to(dev), k, window)
    torch.cuda.synchronize()
    eng.close()
    return {n: v.cpu().numpy() for n, v in out.items()}


def check_tokens(out, ref, k, rows=None):
    """`ref` holds k+1 oracle top entries and the oracle's full log-prob rows (`logp`); `rows` selects GPU rows
    when the oracle scored a sample."""
    sel = (lambda a: a) if rows is None else (lambda a: a[rows])
    for key in ("lse", "target_logprob", "conf"):
        np.testing.assert_allclose(sel(out[key]), ref[key], rtol=0, atol=ABS_TOL, err_msg=key)
    np.testing.assert_allclose(sel(out["entropy"]), ref["entropy"], rtol=REL_TOL, atol=1e-6, err_msg="entropy")
    tv, ti = sel(out["topk_logprob"]), sel(out["topk_index"])
    rv, ri = ref["topk_logprob"], ref["topk_index"]
    np.testing.assert_allclose(tv, rv[:, :k], rtol=0, atol=ABS_TOL, err_msg="topk_logprob")
    assert (np.diff(tv, axis=1) <= 0).all(), "top-k values must be non-increasing"
    # index j must match where it is separated from both oracle neighbours by more than GAP
    n = rv.shape[0]
    gap_below = np.full((n, k), np.inf)
    kk = rv.shape[1]
    gap_below[:, :min(k, kk - 1)] = (rv[:, :-1] - rv[:, 1:])[:, :k]
    gap_above = np.full((n, k), np.inf)
    gap_above[:, 1:] = (rv[:, :-1] - rv[:, 1:])[:, :k - 1]
    must = (gap_below > GAP) & (gap_above > GAP)
    bad = must & (ti != ri[:, :k])
    assert not bad.any(), "top-k index mismatch at %s" % (np.argwhere(bad)[:5],)
    # Where several id sets are acceptable (near-ties), every reported id must still be valid: inside the
    # vocabulary, distinct within its row, and CARRY ITS VALUE -- the oracle's log-prob of that very id is the
    # reported one (so a stale or wrong id cannot hide in a near-tie).  All rows, all j.
    logp = ref["logp"]
    V = logp.shape[1]
    assert (ti >= 0).all() and (ti < V).all(), "top-k id outside [0, V)"
    if k > 1 and n > 0:
        assert (np.diff(np.sort(ti, axis=1), axis=1) != 0).all(), "duplicate top-k id in a row"
    if n > 0:
        carried = np.take_along_axis(logp, ti.astype(np.int64), axis=1)
        worst = np.abs(carried - tv).max()
        assert worst <= ABS_TOL, "a reported top-k id does not carry the reported value (max gap %g)" % worst


def check_seqs(out, ref):
    for key in SEQ_KEYS:
        a, b = out[key], np.asarray(ref[key])
        assert (np.isnan(a) == np.isnan(b)).all(), key
        ok = ~np.isnan(b)
        np.testing.assert_allclose(a[ok], b[ok], rtol=REL_TOL, atol=1e-6, err_msg=key)


def oracle_full(inp, k=None, window=None, targets=None):
    wl = inp["workload"]
    return O.score(inp["H"], inp["W"], inp["targets"] if targets is None else targets, inp["cu_seqlens"],
                   wl.k if k is None else k, wl.window if window is None else window)


# ------------------------------------------------------------------------------------------ small, full
@pytest.mark.parametrize("cg", [1, 2])
def test_tiny_config(cg):
    inp = workloads.make_inputs(workloads.CONFIGS["tiny"])
    out = run_gpu(inp, cta_group=cg)
    ref = oracle_full(inp)
    check_tokens(out, ref, inp["k"])
    check_seqs(out, ref)


SMALL = [
    # several token tiles, ragged T, d not a multiple of 64, V not a multiple of 32 or 256
    dict(name="ragged", d=200, V=1003, B=3, len_lo=100, len_hi=300, k=5, window=16, seed=5, w_std=0.1),
    # several vocab tiles and chunks, planted peaks
    dict(name="mid", d=512, V=5000, B=3, len_lo=200, len_hi=500, k=20, window=64, seed=6, w_std=0.05,
         planted_frac=0.5, planted_scale=3.0, rmsnorm=True),
    # strongly peaked rows: entropy -> 0 is where rel 1e-3 is hardest
    dict(name="peaked", d=256, V=3000, B=2, len_lo=150, len_hi=260, k=20, window=32, seed=8, w_std=0.05,
         planted_frac=0.5, planted_scale=30.0, rmsnorm=True),
    # vocabulary smaller than one tile, tiny d
    dict(name="smallV", d=8, V=40, B=2, len_lo=5, len_hi=40, k=8, window=4, seed=9, w_std=1.0),
]


@pytest.mark.parametrize("spec", SMALL, ids=[s["name"] for s in SMALL])
@pytest.mark.parametrize("cg,chunks,gm", [(2, 0, 0), (1, 0, 0), (2, 3, 2), (1, 2, 1), (2, 1, 8)])
def test_small_shapes_full_parity(spec, cg, chunks, gm):
    inp = workloads.make_inputs(workloads.custom(**spec))
    out = run_gpu(inp, cta_group=cg, num_chunks=chunks, group_m=gm)
    ref = oracle_full(inp)
    check_tokens(out, ref, inp["k"])
    check_seqs(out, ref)


@pytest.mark.parametrize("T,cg", [(1, 2), (7, 1), (64, 2), (128, 1), (300, 2)])
def test_decode_shaped_many_chunks(T, cg):
    """Small T (self-confidence during decode): the planner gives every cluster its
    own slice of the vocabulary (up to 160 chunks per row), merged by the finalize kernel."""
    import paper_2604_07725_b200 as sq
    wl = workloads.custom(name="decode", d=128, V=40000, B=1, len_lo=T, len_hi=T, k=20, window=4, seed=50 + T, w_std=0.1,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    assert sq.plan(wl.d, wl.V, T, 20, 148, cta_group=cg)["num_chunks"] > (32 if T <= 256 else 16)   # 157 vocab tiles: 79 / 53 / 27 chunks
    out = run_gpu(inp, cta_group=cg)
    ref = oracle_full(inp)
    check_tokens(out, ref, 20)
    check_seqs(out, ref)


@pytest.mark.parametrize("k", [1, 5, 8, 9, 20, 21, 32])
def test_every_topk_capacity(k):
    inp = workloads.make_inputs(workloads.custom(name="k", d=64, V=2000, B=2, len_lo=60, len_hi=200, k=k, window=8,
                                                 seed=20 + k, w_std=0.2))
    out = run_gpu(inp)
    ref = oracle_full(inp)
    check_tokens(out, ref, k)
    check_seqs(out, ref)
    assert out["conf"].min() >= math.log(k) - 1e-4        # Jensen bound, reading #2


def test_k_equals_vocab():
    inp = workloads.make_inputs(workloads.custom(name="kV", d=16, V=8, B=1, len_lo=50, len_hi=50, k=8, window=8, seed=3, w_std=1.0))
    out = run_gpu(inp)
    ref = oracle_full(inp)
    check_tokens(out, ref, 8)
    np.testing.assert_allclose(np.exp(out["topk_logprob"].astype(np.float64)).sum(1), 1.0, atol=1e-4)
    for r in range(inp["T"]):
        assert sorted(out["topk_index"][r].tolist()) == list(range(8))


# ------------------------------------------------------------------------------------------ edge cases
def test_empty_short_and_single_token_sequences():
    wl = workloads.custom(name="edge", d=64, V=700, B=6, k=5, window=16, seed=31, w_std=0.2)
    inp = workloads.make_inputs(wl, lengths=[0, 1, 15, 16, 17, 300])     # empty, L=1, L<w, L=w, L=w+1, long
    out = run_gpu(inp)
    ref = oracle_full(inp)
    check_tokens(out, ref, 5)
    check_seqs(out, ref)
    assert np.isnan(out["seq_mean_conf"][0]) and np.isnan(out["seq_min_window_conf"][0])
    assert out["seq_min_window_conf"][1] == pytest.approx(out["conf"][0], rel=1e-6)


@pytest.mark.parametrize("window", [1, 3, 16, 17, 40, 1000])
def test_small_run_sequences_reduced_in_the_finalize_tail(window):
    """Runs of at most 256 tokens (decode-shaped) do kernel 2's work in the finalize kernel's last CTA (two launches):
    empty, L = 1, L < w, L = w, L = w + 1 sequences, invalid targets, a sequence without any valid target; twice on
    one ctx (the CTA counter must be back to zero)."""
    sq = _sq()
    wl = workloads.custom(name="tail", d=64, V=3000, B=8, k=20, window=window, seed=36, w_std=0.2,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl, lengths=[128, 0, 1, 15, 16, 17, 0, 40, 39])   # T = 256
    tg = inp["targets"].clone()
    tg[1:16:2] = -1
    tg[-39:] = wl.V + 7                                                           # the last sequence has no valid target
    dev = torch.device("cuda:0")
    eng = sq.SqScore(wl.d, wl.V, max_tokens=256, max_seqs=9, max_k=20)
    H, W, cu = inp["H"].to(dev), inp["W"].to(dev), inp["cu_seqlens"].to(dev)
    ref = oracle_full(inp, targets=tg.numpy(), window=window)
    for rep in range(2):
        n0 = eng.launch_count()
        out = eng.run(H, W, tg.to(dev), cu, 20, window)
        torch.cuda.synchronize()
        assert eng.launch_count() - n0 == 2
        o = {n: v.cpu().numpy() for n, v in out.items()}
        check_tokens(o, ref, 20)
        check_seqs(o, ref)
        assert np.isnan(o["seq_mean_logprob"][[1, 6, 8]]).all() and np.isfinite(o["seq_mean_entropy"][8])
    # one more token and kernel 2 is a launch of its own again; the results agree
    eng2 = sq.SqScore(wl.d, wl.V, max_tokens=257, max_seqs=9, max_k=20)
    inp3 = workloads.make_inputs(wl, lengths=[128, 0, 1, 15, 16, 17, 0, 40, 40])
    n0 = eng2.launch_count()
    out3 = eng2.run(inp3["H"].to(dev), W, inp3["targets"].to(dev), inp3["cu_seqlens"].to(dev), 20, window)
    torch.cuda.synchronize()
    assert eng2.launch_count() - n0 == 3
    ref3 = oracle_full(inp3, window=window)
    check_seqs({n: v.cpu().numpy() for n, v in out3.items()}, ref3)
    eng.close(); eng2.close()


def test_all_sequences_empty_and_zero_tokens():
    wl = workloads.custom(name="none", d=64, V=300, B=3, k=5, window=4, seed=32)
    inp = workloads.make_inputs(wl, lengths=[0, 0, 0])
    out = run_gpu(inp)
    for key in SEQ_KEYS:
        assert np.isnan(out[key]).all()
    assert out["lse"].shape == (0,)


def test_no_target_rows_are_excluded_from_the_mean():
    wl = workloads.custom(name="notgt", d=64, V=500, B=2, len_lo=40, len_hi=80, k=5, window=8, seed=33, w_std=0.2)
    inp = workloads.make_inputs(wl)
    tg = inp["targets"].clone()
    tg[::3] = -1
    tg[1::7] = wl.V          # == V is also "no target"
    L0 = int(inp["cu_seqlens"][1])
    out = run_gpu(inp, targets=tg)
    ref = oracle_full(inp, targets=tg.numpy())
    check_tokens(out, ref, 5)
    check_seqs(out, ref)
    assert (out["target_logprob"][::3] == 0).all()
    # a sequence whose targets are all invalid has a NaN log-prob mean and finite other aggregates
    tg2 = inp["targets"].clone(); tg2[:L0] = -1
    out2 = run_gpu(inp, targets=tg2)
    assert np.isnan(out2["seq_mean_logprob"][0]) and np.isfinite(out2["seq_mean_logprob"][1])
    assert np.isfinite(out2["seq_mean_entropy"]).all()


def test_targets_on_tile_edges_and_topk_positions():
    V, d = 1100, 64
    cols = [0, 31, 32, 127, 128, 255, 256, 511, 512, 1023, 1024, V - 1]
    T = len(cols) * 11
    g = torch.Generator().manual_seed(4)
    W = (torch.randn(V, d, generator=g) * 0.05).to(torch.bfloat16)
    H = torch.randn(T, d, generator=g)
    tg = torch.tensor([cols[t % len(cols)] for t in range(T)], dtype=torch.int32)
    H = (H / H.norm(dim=1, keepdim=True) * 8 + 40.0 * W[tg.long()].float()).to(torch.bfloat16)   # the target wins top-1
    wl = workloads.custom(name="edges", d=d, V=V, B=1, k=5, window=8)
    inp = {"H": H, "W": W, "targets": tg, "cu_seqlens": torch.tensor([0, T], dtype=torch.int32), "k": 5, "window": 8,
           "workload": wl, "T": T, "B": 1}
    for cg in (1, 2):
        out = run_gpu(inp, cta_group=cg, num_chunks=2)
        ref = oracle_full(inp)
        check_tokens(out, ref, 5)
        assert (out["topk_index"][:, 0] == tg.numpy()).all()
        np.testing.assert_allclose(out["target_logprob"], out["topk_logprob"][:, 0], atol=1e-6)


def test_duplicate_rows_give_bit_identical_outputs():
    wl = workloads.custom(name="dup", d=128, V=3000, B=1, len_lo=600, len_hi=600, k=20, window=8, seed=35, w_std=0.1)
    inp = workloads.make_inputs(wl)
    src = 5
    places = [0, 31, 32, 127, 128, 255, 256, 300, 511, 599]      # different lanes, warps, CTAs of a pair, token tiles
    for t in places:
        inp["H"][t] = inp["H"][src]
        inp["targets"][t] = inp["targets"][src]
    out = run_gpu(inp, num_chunks=3)
    for key in ("lse", "target_logprob", "entropy", "conf", "topk_logprob", "topk_index"):
        for t in places:
            assert (out[key][t] == out[key][src]).all(), (key, t)


# ------------------------------------------------------------------------------------------ closed forms on the GPU
def test_identical_w_rows_closed_form():
    V, d, T = 1500, 64, 300
    g = torch.Generator().manual_seed(2)
    w = (torch.randn(d, generator=g) * 0.3).to(torch.bfloat16)
    W = w.repeat(V, 1).contiguous()
    H = torch.randn(T, d, generator=g).to(torch.bfloat16)
    wl = workloads.custom(name="ident", d=d, V=V, B=1, k=20, window=8)
    inp = {"H": H, "W": W, "targets": torch.randint(0, V, (T,), generator=g, dtype=torch.int32),
           "cu_seqlens": torch.tensor([0, T], dtype=torch.int32), "k": 20, "window": 8, "workload": wl, "T": T, "B": 1}
    out = run_gpu(inp, num_chunks=3)
    lnV = math.log(V)
    z = (H.double() @ w.double()).numpy()
    np.testing.assert_allclose(out["lse"], z + lnV, atol=ABS_TOL)
    np.testing.assert_allclose(out["target_logprob"], -lnV, atol=ABS_TOL)      # BASELINE.json pin
    np.testing.assert_allclose(out["entropy"], lnV, rtol=REL_TOL)              # BASELINE.json pin
    np.testing.assert_allclose(out["topk_logprob"], -lnV, atol=ABS_TOL)
    np.testing.assert_allclose(out["conf"], lnV, atol=ABS_TOL)
    for r in range(0, T, 37):                                                  # ties: any 20 distinct valid ids
        ids = out["topk_index"][r]
        assert len(set(ids.tolist())) == 20 and ids.min() >= 0 and ids.max() < V
    np.testing.assert_allclose(out["seq_mean_entropy"], lnV, rtol=REL_TOL)


@pytest.mark.parametrize("shift", [80.0, -80.0])
def test_large_logit_shift(shift):
    # a constant W column seen by a constant H column shifts every logit by `shift`: catches a
    # missing max-subtraction (exp overflow/underflow in fp32)
    wl = workloads.custom(name="shift", d=64, V=2000, B=1, len_lo=200, len_hi=200, k=5, window=8, seed=37, w_std=0.1)
    inp = workloads.make_inputs(wl)
    inp["H"][:, 63] = 8.0
    inp["W"][:, 63] = shift / 8.0
    out = run_gpu(inp, num_chunks=2)
    ref = oracle_full(inp)
    check_tokens(out, ref, 5)
    check_seqs(out, ref)
    assert np.isfinite(out["lse"]).all() and abs(np.median(out["lse"]) - shift) < 20


# ------------------------------------------------------------------------------------------ full-size configs
def sample_rows(inp, n_planted=136, n_unplanted=136, n_uniform=240, seed=123):
    """Seeded row sample for oracle-A at full size (>= 512 rows, >= 128 planted and >= 128
    unplanted): first/last row, rows next to every sequence boundary, token-tile edges, planted and
    unplanted rows, the rest uniform."""
    T = inp["T"]
    cu = inp["cu_seqlens"].numpy().astype(np.int64)
    rows = {0, T - 1, 127, 128, 255, 256, 257, 511, 512}
    for c in cu[1:-1]:
        rows.update((int(c) - 1, int(c)))
    rng = np.random.default_rng(seed)
    pl = inp["planted"].numpy()
    for mask, n in ((pl, n_planted), (~pl, n_unplanted)):
        idx = np.nonzero(mask)[0]
        assert len(idx) >= n
        rows.update(rng.choice(idx, size=n, replace=False).tolist())
    rows.update(rng.integers(0, T, size=n_uniform).tolist())
    last_tile = (T - 1) // 256 * 256
    rows.update((last_tile, min(T - 1, last_tile + 129)))
    rows = np.array(sorted(r for r in rows if 0 <= r < T), dtype=np.int64)
    assert len(rows) >= 512 and pl[rows].sum() >= 128 and (~pl[rows]).sum() >= 128
    return rows


@pytest.mark.parametrize("name", ["qwen3_4b", "qwen3_8b", "gpt_oss", "qwen3_32b"])
def test_full_size_config_sampled_rows_and_all_sequences(name):
    """BASELINE.json configs 2-5 at full size in the launch configuration bench.py times (default
    planner, CTA pairs): kernel 1 + finalize on >= 512 sampled rows (oracle-A), kernel 2 on every sequence
    (oracle-B applied to the GPU's own per-token outputs), and one whole sequence end to end."""
    sq = _sq()
    wl = workloads.CONFIGS[name]
    inp = workloads.make_inputs(wl)
    out = run_gpu(inp)
    T, k = inp["T"], wl.k
    pln = sq.plan(wl.d, wl.V, T, k, num_sms=torch.cuda.get_device_properties(0).multi_processor_count)
    assert pln["clusters_used"] == pln["num_clusters"], "the launch must use every CTA pair of the device: %s" % (pln,)
    W64 = O.widen(inp["W"])
    tg = inp["targets"].numpy()
    rows = sample_rows(inp)
    for r0 in range(0, len(rows), 64):                 # in batches: the oracle's full log-prob rows are 64 x V fp64
        rb = rows[r0:r0 + 64]
        check_tokens(out, O.token_scores(inp["H"][rb], W64, tg[rb], k), k, rows=rb)
    # properties that hold for every row at any size
    assert np.isfinite(out["lse"]).all()
    assert (out["entropy"] > 0).all() and (out["entropy"] <= math.log(wl.V) * (1 + 1e-4)).all()
    assert (out["target_logprob"] <= 1e-4).all()
    assert (out["conf"] >= math.log(k) - 1e-3).all()
    assert (np.diff(out["topk_logprob"], axis=1) <= 0).all()
    assert (out["target_logprob"] <= out["topk_logprob"][:, 0] + 1e-5).all()
    assert (out["topk_index"] >= 0).all() and (out["topk_index"] < wl.V).all()
    assert (np.diff(np.sort(out["topk_index"], axis=1), axis=1) != 0).all()            # distinct ids in every row
    pl = inp["planted"].numpy()
    if pl.any() and (~pl).any():
        assert out["target_logprob"][pl].mean() > out["target_logprob"][~pl].mean() + 1.0   # planted rows favour the target
    # kernel 2 at full size, isolated: fp64 reduction oracle on the GPU's per-token outputs
    seq_ref = O.sequence_scores(out["target_logprob"], out["entropy"], out["conf"], inp["cu_seqlens"].numpy(), wl.window)
    check_seqs(out, seq_ref)
    # one whole sequence end to end from H and W (the shortest one)
    cu = inp["cu_seqlens"].numpy().astype(np.int64)
    b = int(np.argmin(np.diff(cu)))
    lo, hi = int(cu[b]), int(cu[b + 1])
    assert 0 < hi - lo <= 4096, "the shortest sequence of %s has %d rows: too long for the end-to-end oracle leg" % (name, hi - lo)
    parts = []
    for r0 in range(lo, hi, 64):
        r1 = min(hi, r0 + 64)
        ref = O.token_scores(inp["H"][r0:r1], W64, tg[r0:r1], k)
        check_tokens(out, ref, k, rows=np.arange(r0, r1))
        parts.append({key: ref[key] for key in ("target_logprob", "entropy", "conf")})
    full = {key: np.concatenate([p[key] for p in parts]) for key in ("target_logprob", "entropy", "conf")}
    e2e = O.sequence_scores(full["target_logprob"], full["entropy"], full["conf"], [0, hi - lo], wl.window)
    for key in SEQ_KEYS:
        np.testing.assert_allclose(out[key][b], e2e[key][0], rtol=REL_TOL, err_msg=key)


# ------------------------------------------------------------------------------------------ kernel 2 alone
def _reduce_all_forms(sq, make_engine, call, stream_form="stream"):
    """Kernel 2 forced into its single-launch form (sq_score_config.debug_flags bit 6), its three-launch tile form (bit 5) and its
    streaming form (bit 8; `stream_form` = "tiles" where the window is too wide for it and the tile form takes over).  The
    two tile forms must agree bit for bit; returns (single-launch outputs, streaming outputs) -- the caller checks both
    against the oracle."""
    import os
    outs = []
    for dbg in ("64", "32", "256"):
        eng = make_engine(int(dbg))
        n0 = eng.launch_count()
        o = call(eng)
        torch.cuda.synchronize()
        assert eng.launch_count() - n0 == {"64": 1, "32": 3, "256": 2 if stream_form == "stream" else 3}[dbg]
        assert eng.reduce_form() == {"64": "fused", "32": "tiles", "256": stream_form}[dbg]
        outs.append({n: v.cpu().numpy() for n, v in o.items()})
        o2 = call(eng)                                   # a second run on the same ctx: nothing is left over from the first
        torch.cuda.synchronize()
        for n in o:
            np.testing.assert_array_equal(outs[-1][n], o2[n].cpu().numpy())
        eng.close()
    for n in outs[0]:
        np.testing.assert_array_equal(outs[0][n], outs[1][n])
    return outs[0], outs[2]


@pytest.mark.parametrize("window", [1, 2, 3, 16, 511, 512, 513, 2048, 4096, 4097, 8191, 8192, 8193, 8195, 12290, 100000])
def test_reduce_kernel_alone(window):
    sq = _sq()
    lens = [1, 2, 511, 512, 513, 0, 4095, 4096, 4097, 8192, 9000, 20000, 3, 1025]
    g = torch.Generator().manual_seed(77)
    T = sum(lens)
    cu = torch.tensor(np.concatenate([[0], np.cumsum(lens)]), dtype=torch.int32)
    lp = -(torch.rand(T, generator=g) * 12); en = torch.rand(T, generator=g) * 11; cf = 3 + torch.rand(T, generator=g) * 12
    cf[30000:30040] = 0.5                      # a dip the minimum window must find
    dev = torch.device("cuda:0")
    a = [x.to(dev) for x in (lp, en, cf, cu)]
    out, out_s = _reduce_all_forms(sq, lambda dbg: sq.SqScore(64, 1000, max_tokens=T, max_seqs=len(lens), max_k=5, reduce_only=True, debug_flags=dbg),
                                   lambda eng: eng.reduce(a[0], a[1], a[2], a[3], window),
                                   stream_form="stream" if 128 <= window <= 2048 else "tiles")
    ref = O.sequence_scores(lp.numpy(), en.numpy(), cf.numpy(), cu.numpy(), window)
    check_seqs(out, ref)
    check_seqs(out_s, ref)


@pytest.mark.parametrize("offset", [0, 1, 3])
@pytest.mark.parametrize("with_targets", [False, True])
@pytest.mark.parametrize("dbg", [None, "256"], ids=["default", "streaming"])
def test_reduce_alignment_targets_and_array_end(offset, with_targets, dbg):
    """Kernel 2's 16-byte-load path against its scalar path: arrays that start `offset` floats into an allocation
    (unaligned -> scalar loads), a total length that is not a multiple of 4 (the last vector would cross the end of
    the arrays), sequences that start and end inside a block, windows with every residue mod 4, invalid targets."""
    sq = _sq()
    lens = [5, 8190, 3, 8193, 16384, 1, 0, 12289, 4094, 7]          # T = 49165, odd
    T = sum(lens)
    g = torch.Generator().manual_seed(78 + offset)
    cu = torch.tensor(np.concatenate([[0], np.cumsum(lens)]), dtype=torch.int32)
    lp = -(torch.rand(T, generator=g) * 12); en = torch.rand(T, generator=g) * 11; cf = 3 + torch.rand(T, generator=g) * 12
    cf[T - 600:T - 560] = 0.25                                       # a dip close to the end of the arrays
    tg = torch.randint(0, 1000, (T,), generator=g, dtype=torch.int32)
    tg[torch.rand(T, generator=g) < 0.2] = -1
    tg[8195:8195 + 8193] = 5000                                      # a whole sequence without a valid target
    dev = torch.device("cuda:0")
    def place(x):                                                    # the same values at an `offset`-element misalignment
        buf = torch.empty(T + 8, dtype=x.dtype, device=dev)
        buf[offset:offset + T] = x.to(dev)
        return buf[offset:offset + T]
    import os
    eng = sq.SqScore(64, 1000, max_tokens=T, max_seqs=len(lens), max_k=5, reduce_only=True, debug_flags=int(dbg or 0))
    valid = ((tg >= 0) & (tg < 1000)).numpy() if with_targets else None
    for window in (1, 6, 1023, 2047, 2048, 2049, 2050, 8192, 8195, 30000):
        out = eng.reduce(place(lp), place(en), place(cf), cu.to(dev), window, targets=place(tg) if with_targets else None)
        torch.cuda.synchronize()
        assert eng.reduce_form() == (("stream" if offset == 0 and 128 <= window <= 2048 else "tiles") if dbg else "fused")
        ref = O.sequence_scores(lp.numpy(), en.numpy(), cf.numpy(), cu.numpy(), window, target_valid=valid)
        check_seqs({n: v.cpu().numpy() for n, v in out.items()}, ref)
    eng.close()


def test_reduce_many_sequences():
    sq = _sq()
    r = workloads.reduction_inputs(3000, 1, 3000, seed=5)
    dev = torch.device("cuda:0")
    a = [r[n].to(dev) for n in ("target_logprob", "entropy", "conf", "cu_seqlens")]
    out, out_s = _reduce_all_forms(sq, lambda dbg: sq.SqScore(64, 1000, max_tokens=r["T"], max_seqs=r["B"], max_k=5, reduce_only=True, debug_flags=dbg),
                                   lambda eng: eng.reduce(a[0], a[1], a[2], a[3], 256))
    ref = O.sequence_scores(r["target_logprob"].numpy(), r["entropy"].numpy(), r["conf"].numpy(), r["cu_seqlens"].numpy(), 256)
    check_seqs(out, ref)
    check_seqs(out_s, ref)


@pytest.mark.parametrize("dbg,form,window", [(None, "stream", 130), ("32", "tiles", 7), (None, "tiles", 7)], ids=["streaming", "three-launch", "narrow-window"])
def test_reduce_more_sequences_than_the_single_launch_form_holds(dbg, form, window):
    """B = 13 000 > 12 287 short sequences (many per 256-token range, empty ones among them): more than one wave, so the
    streaming form runs by default; forced off, the tile table no longer fits in shared memory and the three-launch form
    runs."""
    import os
    sq = _sq()
    r = workloads.reduction_inputs(13000, 0, 40, seed=6)
    dev = torch.device("cuda:0")
    eng = sq.SqScore(64, 1000, max_tokens=r["T"], max_seqs=r["B"], max_k=5, reduce_only=True, debug_flags=int(dbg or 0))
    out = eng.reduce(r["target_logprob"].to(dev), r["entropy"].to(dev), r["conf"].to(dev), r["cu_seqlens"].to(dev), window)
    torch.cuda.synchronize()
    assert eng.launch_count() == (2 if form == "stream" else 3) and eng.reduce_form() == form
    ref = O.sequence_scores(r["target_logprob"].numpy(), r["entropy"].numpy(), r["conf"].numpy(), r["cu_seqlens"].numpy(), window)
    check_seqs({n: v.cpu().numpy() for n, v in out.items()}, ref)
    eng.close()


def test_reduce_streaming_form_many_sequences_per_range_and_one_long_sequence():
    """The streaming form's fold: many sequences inside one 256-token range, sequences that start exactly on range and
    block boundaries, empty sequences at position 0, in the middle and at the
    end, one sequence that spans many blocks, windows of every residue mod 4 and below / at / above the range size, up to
    RS_WMAX."""
    import os
    sq = _sq()
    lens = [0, 0] + [1] * 70 + [186, 256, 0, 512, 4096 - 1280 + 256, 0, 4096, 30011] + [3] * 40 + [2, 0, 0]
    T = sum(lens)
    g = torch.Generator().manual_seed(79)
    cu = torch.tensor(np.concatenate([[0], np.cumsum(lens)]), dtype=torch.int32)
    lp = -(torch.rand(T, generator=g) * 12); en = torch.rand(T, generator=g) * 11; cf = 3 + torch.rand(T, generator=g) * 12
    cf[20000:20100] = 0.5
    dev = torch.device("cuda:0")
    eng = sq.SqScore(64, 1000, max_tokens=T, max_seqs=len(lens), max_k=5, reduce_only=True, debug_flags=int("256" or 0))
    for window in (128, 129, 130, 131, 255, 256, 257, 1000, 2047, 2048):
        out = eng.reduce(lp.to(dev), en.to(dev), cf.to(dev), cu.to(dev), window)
        torch.cuda.synchronize()
        assert eng.reduce_form() == "stream"
        ref = O.sequence_scores(lp.numpy(), en.numpy(), cf.numpy(), cu.numpy(), window)
        check_seqs({n: v.cpu().numpy() for n, v in out.items()}, ref)
    eng.close()


def test_reduce_streaming_form_every_sequence_empty_then_a_normal_call():
    """Every warp of the fold kernel leaves early (all sequences empty although T > 0: a cu_seqlens the caller got wrong):
    NaNs everywhere, and the next call on the ctx -- whose stream kernel overwrites the same records -- is correct, i.e. the
    fold grid did not finish ahead of the stream kernel it was launched behind."""
    import os
    sq = _sq()
    r = workloads.reduction_inputs(300, 100, 900, seed=9)
    dev = torch.device("cuda:0")
    eng = sq.SqScore(64, 1000, max_tokens=r["T"], max_seqs=r["B"], max_k=5, reduce_only=True, debug_flags=int("256" or 0))
    a = [r[n].to(dev) for n in ("target_logprob", "entropy", "conf", "cu_seqlens")]
    empty = eng.reduce(a[0], a[1], a[2], torch.zeros_like(a[3]), 256)
    out = eng.reduce(a[0], a[1], a[2], a[3], 256)                 # enqueued right behind it, no host sync between
    torch.cuda.synchronize()
    assert eng.reduce_form() == "stream"
    for n in SEQ_KEYS:
        assert torch.isnan(empty[n]).all(), n
    ref = O.sequence_scores(r["target_logprob"].numpy(), r["entropy"].numpy(), r["conf"].numpy(), r["cu_seqlens"].numpy(), 256)
    check_seqs({n: v.cpu().numpy() for n, v in out.items()}, ref)
    eng.close()


def test_small_run_with_an_inconsistent_cu_seqlens_stays_inside_its_arrays():
    """cu_seqlens is device data nobody checks (sq_score_positions writes an inconsistent one when its status is non-zero).
    In a run of at most 256 tokens the finalize tail clamps it into [0, T]: a last entry far beyond T, and a negative
    one, neither overrun the 257-entry prefix in shared memory nor the per-token arrays; sequences whose bounds are
    sound keep their values, a clamped one is reduced over the tokens that exist."""
    sq = _sq()
    wl = workloads.custom(name="badcu", d=64, V=3000, B=3, k=20, window=16, seed=37, w_std=0.2,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl, lengths=[100, 60, 96])                        # T = 256
    dev = torch.device("cuda:0")
    eng = sq.SqScore(wl.d, wl.V, max_tokens=256, max_seqs=3, max_k=20)
    H, W, tg = inp["H"].to(dev), inp["W"].to(dev), inp["targets"].to(dev)
    good = eng.run(H, W, tg, inp["cu_seqlens"].to(dev), 20, 16)
    torch.cuda.synchronize()
    assert eng.reduce_form() == "tail"
    bad = eng.run(H, W, tg, torch.tensor([0, 100, 160, 100000], dtype=torch.int32, device=dev), 20, 16)   # end >> T
    neg = eng.run(H, W, tg, torch.tensor([-500, 100, 160, 256], dtype=torch.int32, device=dev), 20, 16)   # start < 0
    torch.cuda.synchronize()
    again = eng.run(H, W, tg, inp["cu_seqlens"].to(dev), 20, 16)
    torch.cuda.synchronize()
    for n in SEQ_KEYS:
        assert torch.equal(bad[n], good[n]), n            # [160, 100000) clamps to [160, 256): the sequence that exists
        assert torch.equal(neg[n], good[n]), n            # [-500, 100) clamps to [0, 100)
        assert torch.equal(again[n], good[n]), n
    eng.close()


def test_scoring_pipeline_takes_the_streaming_form_for_many_sequences():
    """sq_score_run on a population of 2 300 candidates (more than one wave of kernel-2 tiles): kernel 1 -> finalize ->
    streaming form of kernel 2, chained by programmatic dependent launches.  The per-sequence outputs against oracle-B
    (fp64 reductions of the GPU's own per-token outputs), invalid targets included, and a sample of rows against oracle-A."""
    sq = _sq()
    wl = workloads.custom(name="many", d=64, V=512, B=2300, len_lo=90, len_hi=420, k=5, window=128, seed=88, w_std=0.05,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    tg = inp["targets"].clone()
    tg[torch.rand(inp["T"], generator=torch.Generator().manual_seed(3)) < 0.1] = -1
    dev = torch.device("cuda:0")
    eng = sq.SqScore(wl.d, wl.V, max_tokens=inp["T"], max_seqs=inp["B"], max_k=wl.k)
    out = eng.run(inp["H"].to(dev), inp["W"].to(dev), tg.to(dev), inp["cu_seqlens"].to(dev), wl.k, wl.window)
    torch.cuda.synchronize()
    assert eng.reduce_form() == "stream"
    out2 = eng.run(inp["H"].to(dev), inp["W"].to(dev), tg.to(dev), inp["cu_seqlens"].to(dev), wl.k, wl.window)
    torch.cuda.synchronize()
    for n in SEQ_KEYS:
        assert torch.equal(out[n], out2[n], ) or (torch.isnan(out[n]) == torch.isnan(out2[n])).all()
    eng.close()
    out = {n: v.cpu().numpy() for n, v in out.items()}
    valid = ((tg >= 0) & (tg < wl.V)).numpy()
    seq_ref = O.sequence_scores(out["target_logprob"], out["entropy"], out["conf"], inp["cu_seqlens"].numpy(), wl.window, target_valid=valid)
    check_seqs(out, seq_ref)
    rows = np.unique(np.random.default_rng(8).integers(0, inp["T"], 300))
    rows = rows[valid[rows]]
    ref = O.token_scores(inp["H"][rows], O.widen(inp["W"]), tg.numpy()[rows], wl.k)
    check_tokens(out, ref, wl.k, rows=rows)


@pytest.mark.parametrize("d,V,B,lo,hi,gm", [(256, 3000, 6, 700, 1100, 0), (200, 1003, 9, 500, 900, 3), (512, 5000, 4, 1500, 2500, 6)])
def test_quad_scheduling_with_w_multicast(d, V, B, lo, hi, gm):
    """sq_score_config.cluster4 = 1 (by default only runs of more than 200 000 tokens -- the full-size qwen3_32b test --
    take this path): runs of more than 4096 tokens are scheduled in quads of four CTAs that
    the device places as clusters of 4 (W boxes multicast to both CTA pairs) or, where it cannot, as two pairs; 512-row
    token tiles, ragged T, d and V.  Same tolerances against the oracle; bf16 and the FP8 variant."""
    import os
    sq = _sq()
    wl = workloads.custom(name="quad", d=d, V=V, B=B, len_lo=lo, len_hi=hi, k=20, window=64, seed=d + V, w_std=0.05,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    assert inp["T"] > 4096
    dev = torch.device("cuda:0")
    eng = sq.SqScore(d, V, max_tokens=inp["T"], max_seqs=B, max_k=20, group_m=gm, cluster4=1)
    H, W, tg, cu = (inp[n].to(dev) for n in ("H", "W", "targets", "cu_seqlens"))
    out = eng.run(H, W, tg, cu, 20, 64)
    torch.cuda.synchronize()
    o = {n: v.cpu().numpy() for n, v in out.items()}
    ref = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], 20, 64)
    check_tokens(o, ref, 20); check_seqs(o, ref)
    if d % 16 == 0:
        Hq, hs = eng.quantize_fp8(H, False); Wq, ws = eng.quantize_fp8(W, True)
        o8 = eng.run_fp8(Hq, hs, Wq, ws, tg, cu, 20, 64)
        torch.cuda.synchronize()
        ref8 = O.score(O.dequantize_fp8(Hq.cpu().numpy(), hs.cpu().numpy()), O.dequantize_fp8(Wq.cpu().numpy(), ws.cpu().numpy()),
                       inp["targets"], inp["cu_seqlens"], 20, 64)
        o8 = {n: v.cpu().numpy() for n, v in o8.items()}
        check_tokens(o8, ref8, 20); check_seqs(o8, ref8)
    eng.close()


# ------------------------------------------------------------------------------------------ API behaviour
def test_run_host_matches_run_and_null_per_token_outputs():
    sq = _sq()
    inp = workloads.make_inputs(workloads.custom(name="host", d=128, V=3000, B=3, len_lo=100, len_hi=400, k=20, window=32, seed=41, w_std=0.1))
    dev = torch.device("cuda:0")
    eng = sq.SqScore(128, 3000, max_tokens=inp["T"], max_seqs=3, max_k=20, staging=True)
    W = inp["W"].to(dev)
    out = eng.run(inp["H"].to(dev), W, inp["targets"].to(dev), inp["cu_seqlens"].to(dev), 20, 32)
    out_seq_only = eng.run(inp["H"].to(dev), W, inp["targets"].to(dev), inp["cu_seqlens"].to(dev), 20, 32, per_token=False, topk=False)
    host = torch.empty(12, dtype=torch.float32).pin_memory()
    eng.run_host(inp["H"].pin_memory(), W, inp["targets"].pin_memory(), inp["cu_seqlens"].pin_memory(), 20, 32, host)
    torch.cuda.synchronize()
    dev_seq = torch.cat([out[n] for n in SEQ_KEYS]).cpu()
    assert torch.equal(dev_seq, host)
    assert torch.equal(dev_seq, torch.cat([out_seq_only[n] for n in SEQ_KEYS]).cpu())
    assert eng.launch_count() == 9      # kernel 1, finalize, kernel 2 (single launch) per run
    eng.close()


@pytest.mark.parametrize("T", [2048 * 3 + 17, 2048 * 256 + 5000])
def test_run_host_streams_h_in_blocks(T):
    """sq_score_run_host with several arrival flags (and, for the large T, blocks of 4096 rows because a run uses at
    most 256 flags): H lands while kernel 1 runs; the result must be bit-equal to the device-resident path, twice in a
    row on the same ctx (the staging buffers and flags are reused)."""
    sq = _sq()
    B = 7
    wl = workloads.custom(name="host_blocks", d=64, V=700, B=B, len_lo=1, len_hi=2, k=5, window=64, seed=43, w_std=0.2)
    base = T // B
    lens = [base] * (B - 1) + [T - base * (B - 1)]
    inp = workloads.make_inputs(wl, lengths=lens)
    dev = torch.device("cuda:0")
    eng = sq.SqScore(wl.d, wl.V, max_tokens=T, max_seqs=B, max_k=5, staging=True)
    W = inp["W"].to(dev)
    out = eng.run(inp["H"].to(dev), W, inp["targets"].to(dev), inp["cu_seqlens"].to(dev), 5, 64, per_token=False, topk=False)
    torch.cuda.synchronize()
    dev_seq = torch.cat([out[n] for n in SEQ_KEYS]).cpu()
    Hp, tp, cp = inp["H"].pin_memory(), inp["targets"].pin_memory(), inp["cu_seqlens"].pin_memory()
    for _ in range(2):
        host = torch.full((4 * B,), float("nan")).pin_memory()
        eng.run_host(Hp, W, tp, cp, 5, 64, host)
        torch.cuda.synchronize()
        assert torch.equal(dev_seq, host)
    eng.close()


def test_no_run_call_allocates_and_staging_is_a_create_time_choice():
    """`run` does no allocation.  Device memory in use (cudaMemGetInfo) is read after create and after the
    FIRST call of every run form: it must not move.  Without SQ_FLAG_STAGING, run_host and run_x refuse to run."""
    sq = _sq()
    wl = workloads.custom(name="noalloc", d=256, V=5000, B=4, len_lo=300, len_hi=900, k=20, window=32, seed=45, w_std=0.1)
    inp = workloads.make_inputs(wl)
    pre = workloads.prepare_inputs(wl, query_lo=1, query_hi=20)
    dev = torch.device("cuda:0")
    T, B = inp["T"], inp["B"]
    # every tensor the calls touch exists before the measurement starts
    H, W, tg, cu = (inp[n].to(dev) for n in ("H", "W", "targets", "cu_seqlens"))
    Hp, tp, cp = inp["H"].pin_memory(), inp["targets"].pin_memory(), inp["cu_seqlens"].pin_memory()
    host = torch.empty(4 * B).pin_memory()
    X, gain, ptg = pre["X"].to(dev), pre["gain"].to(dev), pre["targets"].to(dev)
    pos_l, cu_l = sq.trajectory_positions(pre["query_lens"].tolist(), pre["traj_lens"].tolist())
    pos = torch.tensor(pos_l, dtype=torch.int32, device=dev); pcu = torch.tensor(cu_l, dtype=torch.int32, device=dev)
    qd, nd = pre["query_lens"].to(torch.int32).to(dev), pre["traj_lens"].to(torch.int32).to(dev)
    st = torch.empty(sq.shard_state_bytes(T, 20) // 4, device=dev)
    Tm = max(T, pre["T"])
    eng = sq.SqScore(wl.d, wl.V, max_tokens=Tm, max_seqs=B, max_k=20, staging=True)
    out = eng._alloc_out(T, B, 20, dev, True, True)
    outx = eng._alloc_out(pre["T"], pre["B"], 20, dev, True, True)
    pos2 = torch.empty(pre["T"], dtype=torch.int32, device=dev); cu2 = torch.empty(pre["B"] + 1, dtype=torch.int32, device=dev)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(0)[0]
    eng.run(H, W, tg, cu, 20, 32, out=out)
    eng.run_host(Hp, W, tp, cp, 20, 32, host)
    eng.run_x(X, pos, gain, 1e-6, W, ptg, pcu, 20, 32, out=outx)
    eng.run_shard(H, W[:2048], 0, tg, 20, out=st)
    eng.neutral_shard_state(T, 20, out=st)
    eng._check(eng._L.sq_score_positions(eng._h, qd.data_ptr(), nd.data_ptr(), pre["B"], pre["T"], pos2.data_ptr(), cu2.data_ptr(), None,
                                         torch.cuda.current_stream().cuda_stream))
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] == free0, "a run* call allocated device memory"
    assert torch.equal(pos2, pos) and torch.equal(cu2, pcu)
    eng.close()
    plain = sq.SqScore(wl.d, wl.V, max_tokens=Tm, max_seqs=B, max_k=20)
    for call in (lambda: plain.run_host(Hp, W, tp, cp, 20, 32, host), lambda: plain.run_x(X, pos, gain, 1e-6, W, ptg, pcu, 20, 32, out=outx)):
        with pytest.raises(sq.SqScoreError) as ei:
            call()
        assert ei.value.code == sq.ERR_INVALID_ARG and "SQ_FLAG_STAGING" in str(ei.value)
    plain.close()


def test_run_is_cuda_graph_capturable():
    """sq_score_run enqueues only stream work (no allocation, no host sync), so a decode-shaped scoring step can be
    captured once into a CUDA graph and replayed: results bit-equal to the eager call, also after the inputs change."""
    sq = _sq()
    wl = workloads.custom(name="graph", d=256, V=20000, B=2, len_lo=30, len_hi=34, k=20, window=8, seed=91, w_std=0.1,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    dev = torch.device("cuda:0")
    T, B = inp["T"], inp["B"]
    eng = sq.SqScore(wl.d, wl.V, max_tokens=T, max_seqs=B, max_k=20)
    H = inp["H"].to(dev); W = inp["W"].to(dev); tg = inp["targets"].to(dev); cu = inp["cu_seqlens"].to(dev)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        eager = eng.run(H, W, tg, cu, 20, 8, stream=st)
        st.synchronize()
        ref1 = {n: v.clone() for n, v in eager.items()}
        out = {n: torch.empty_like(v) for n, v in eager.items()}
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            eng.run(H, W, tg, cu, 20, 8, stream=st, out=out)
        for _ in range(3):
            g.replay()
        st.synchronize()
        for n in ref1:
            assert torch.equal(out[n], ref1[n]) or (torch.isnan(out[n]) == torch.isnan(ref1[n])).all(), n
        H.copy_(torch.roll(H, 1, 0))               # new hidden states in the same buffer
        g.replay(); st.synchronize()
        eager2 = eng.run(H, W, tg, cu, 20, 8, stream=st)
        st.synchronize()
        for n in eager2:
            assert torch.equal(out[n], eager2[n]), n
        assert not torch.equal(out["lse"], ref1["lse"])
    eng.close()


def test_run_rejects_bad_arguments():
    sq = _sq()
    dev = torch.device("cuda:0")
    eng = sq.SqScore(64, 1000, max_tokens=128, max_seqs=2, max_k=5)
    H = torch.zeros(128, 64, dtype=torch.bfloat16, device=dev); W = torch.zeros(1000, 64, dtype=torch.bfloat16, device=dev)
    tg = torch.zeros(128, dtype=torch.int32, device=dev); cu = torch.tensor([0, 64, 128], dtype=torch.int32, device=dev)
    for kw in (dict(k=6), dict(k=0), dict(window=0)):
        args = dict(k=5, window=4); args.update(kw)
        with pytest.raises(sq.SqScoreError) as ei:
            eng.run(H, W, tg, cu, args["k"], args["window"])
        assert ei.value.code == sq.ERR_INVALID_ARG
    Hbig = torch.zeros(256, 64, dtype=torch.bfloat16, device=dev)
    with pytest.raises(sq.SqScoreError):
        eng.run(Hbig, W, torch.zeros(256, dtype=torch.int32, device=dev), cu, 5, 4)
    with pytest.raises(sq.SqScoreError):
        # H shifted by 8 bytes: not 16-byte aligned
        eng.run(H.view(-1)[4:4 + 64 * 100].view(100, 64), W, tg[:100], torch.tensor([0, 100], dtype=torch.int32, device=dev), 5, 4)
    out = eng.run(H, W, tg, cu, 5, 4)      # the ctx is still usable after errors
    torch.cuda.synchronize()
    assert np.isfinite(out["lse"].cpu().numpy()).all()
    eng.close()
