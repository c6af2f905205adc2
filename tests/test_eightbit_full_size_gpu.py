"""The 8-bit variants against the fp64 oracle AT THE SIZE bench.py TIMES THEM (`fp8_variant` / `mx_variant`: the whole
qwen3_8b batch, default planner, every CTA pair, 27 batches of token tiles, region barriers), and the FP8 kernel in the
quad-scheduled form that runs of more than 200 000 tokens take by default.  The small-shape tests (tests/test_fp8_gpu.py,
tests/test_mx_gpu.py) reach none of those launch configurations.

As there, parity is judged on the QUANTISED operands: the oracle scores the dequantised codes (FP8: the codes and scales
the device quantiser wrote, itself checked against the fp64 definition in test_fp8_gpu.py; MX: the oracle's own
quantisation, which the device's must equal bit for bit on the rows compared) -- PAPER.md:681-692 (very large scorers),
SURVEY.md section 8(f)-4.  Only the sampled rows of H are dequantised; W once (5 GB of fp64 on the host)."""
import math

import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O
from test_parity_gpu import SEQ_KEYS, REL_TOL, check_seqs, check_tokens, sample_rows

pytestmark = pytest.mark.gpu
DEV = torch.device("cuda:0")


def _sq():
    import paper_2604_07725_b200 as sq
    return sq


def _run_variant(variant, inp, expect_cta_group):
    """-> (outputs as numpy, dequantised W fp64, function rows -> dequantised H rows fp64)."""
    sq = _sq()
    wl = inp["workload"]
    eng = sq.SqScore(wl.d, wl.V, max_tokens=inp["T"], max_seqs=inp["B"], max_k=wl.k)
    H, W = inp["H"].to(DEV), inp["W"].to(DEV)
    tg, cu = inp["targets"].to(DEV), inp["cu_seqlens"].to(DEV)
    if variant == "fp8":
        Hq, hs = eng.quantize_fp8(H, False)
        Wq, ws = eng.quantize_fp8(W, True)
        out = eng.run_fp8(Hq, hs, Wq, ws, tg, cu, wl.k, wl.window)
        torch.cuda.synchronize()
        Wd = O.dequantize_fp8(Wq.cpu().numpy(), ws.cpu().numpy())
        hq_host, hs_host = Hq.cpu().numpy(), hs.cpu().numpy()
        h_rows = lambda rb: O.dequantize_fp8(hq_host[rb], hs_host[rb])
    else:
        Hq, hsf = eng.quantize_mx(H, sq.MX_OPERAND_H)
        Wq, wsf = eng.quantize_mx(W, sq.MX_OPERAND_W)
        out = eng.run_mx(Hq, hsf, Wq, wsf, tg, cu, wl.k, wl.window)
        torch.cuda.synchronize()
        table = O.e4m3_values()
        codes_w, exps_w = O.quantize_mx(inp["W"])
        wrows = np.unique(np.concatenate([[0, 223, 224, wl.V - 1], np.random.default_rng(5).integers(0, wl.V, 400)]))
        np.testing.assert_array_equal(table[Wq.cpu().numpy()[wrows]], table[codes_w[wrows]])   # (-0 and +0 are one value)
        Wd = O.dequantize_mx(codes_w, exps_w)
        hq_host = Hq.cpu().numpy()

        def h_rows(rb):
            codes, exps = O.quantize_mx(inp["H"][rb])
            np.testing.assert_array_equal(table[hq_host[rb]], table[codes])      # the rows compared are the rows scored
            return O.dequantize_mx(codes, exps)
    pln = eng.last_plan()
    assert pln["cta_group"] == expect_cta_group, pln
    if expect_cta_group == 2:
        assert pln["clusters_used"] == pln["num_clusters"], "the launch must use every CTA pair of the device: %s" % (pln,)
    del H, W, Hq, Wq
    eng.close()
    return {n: v.cpu().numpy() for n, v in out.items()}, Wd, h_rows


def _check_run(out, inp, Wd, h_rows, rows):
    wl = inp["workload"]
    k, tg = wl.k, inp["targets"].numpy()
    for r0 in range(0, len(rows), 64):                     # the oracle's full log-prob rows are 64 x V fp64 per batch
        rb = rows[r0:r0 + 64]
        check_tokens(out, O.token_scores(h_rows(rb), Wd, tg[rb], k), k, rows=rb)
    # properties that hold for every row at any size
    assert np.isfinite(out["lse"]).all()
    assert (out["entropy"] > 0).all() and (out["entropy"] <= math.log(wl.V) * (1 + 1e-4)).all()
    assert (out["target_logprob"] <= 1e-4).all() and (out["conf"] >= math.log(k) - 1e-3).all()
    assert (np.diff(out["topk_logprob"], axis=1) <= 0).all()
    assert (out["topk_index"] >= 0).all() and (out["topk_index"] < wl.V).all()
    assert (np.diff(np.sort(out["topk_index"], axis=1), axis=1) != 0).all()
    # kernel 2 on every sequence: the fp64 reduction oracle on the GPU's own per-token outputs
    check_seqs(out, O.sequence_scores(out["target_logprob"], out["entropy"], out["conf"], inp["cu_seqlens"].numpy(), wl.window))


@pytest.mark.parametrize("variant", ["fp8", "mx"])
def test_eightbit_full_size_qwen3_8b_sampled_rows(variant):
    wl = workloads.CONFIGS["qwen3_8b"]
    inp = workloads.make_inputs(wl)
    out, Wd, h_rows = _run_variant(variant, inp, expect_cta_group=2)
    rows = sample_rows(inp)                                # >= 512 rows, as the bf16 full-size test
    _check_run(out, inp, Wd, h_rows, rows)
    # the shortest sequence end to end from the quantised operands
    cu = inp["cu_seqlens"].numpy().astype(np.int64)
    b = int(np.argmin(np.diff(cu)))
    lo, hi = int(cu[b]), int(cu[b + 1])
    assert 0 < hi - lo <= 4096
    parts = []
    tg = inp["targets"].numpy()
    for r0 in range(lo, hi, 64):
        rb = np.arange(r0, min(hi, r0 + 64))
        ref = O.token_scores(h_rows(rb), Wd, tg[rb], wl.k)
        check_tokens(out, ref, wl.k, rows=rb)
        parts.append({key: ref[key] for key in ("target_logprob", "entropy", "conf")})
    full = {key: np.concatenate([p[key] for p in parts]) for key in ("target_logprob", "entropy", "conf")}
    e2e = O.sequence_scores(full["target_logprob"], full["entropy"], full["conf"], [0, hi - lo], wl.window)
    for key in SEQ_KEYS:
        np.testing.assert_allclose(out[key][b], e2e[key][0], rtol=REL_TOL, err_msg=key)


def test_fp8_run_of_more_than_200000_tokens_takes_the_quad_kernel_by_default():
    """No environment switch: T > 200 000 alone selects quad scheduling with W multicast (sq_score_last_plan says so), in
    FP8 -- launch_fused<2, CAP, MODE_F8, 4>, which the small tests only reach with sq_score_config.cluster4 = 1."""
    wl = workloads.custom(name="fp8_quad", d=1024, V=50304, B=64, len_lo=2900, len_hi=3700, k=20, window=256, seed=91,
                          w_std=0.03, planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    assert inp["T"] > 200000
    out, Wd, h_rows = _run_variant("fp8", inp, expect_cta_group=4)
    rows = sample_rows(inp)
    _check_run(out, inp, Wd, h_rows, rows)
