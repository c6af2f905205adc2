"""GPU parity of the block-scaled (MX) variant: e4m3 elements, one power-of-two scale per 32 elements of a row, consumed
by tcgen05.mma.kind::mxf8f6f4.block_scale (the widening after SURVEY 8(f)-4; reading #26).

sq_score_quantize_mx is exact arithmetic (exponent from the block maximum, scaling by powers of two, one rounding to
e4m3), so its codes and exponents must equal the oracle's definition (oracle.quantize_mx, pinned by brute force in
tests/test_oracle_mx_pins.py) BIT FOR BIT -- no slack, unlike the per-tensor FP8 variant.  The scale bytes come back in
the layout the tensor core's copy engine wants; `sf_offsets` below restates the header's formula (pure indexing).
sq_score_run_mx meets the path's tolerances against the fp64 oracle evaluated on the dequantised operands (exact in
fp64).  The distance to the bf16 scores is measured next to the per-tensor FP8 variant's."""
import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O
from test_parity_gpu import check_seqs, check_tokens

pytestmark = pytest.mark.gpu
DEV = torch.device("cuda:0")


def _sq():
    import paper_2604_07725_b200 as sq
    return sq


def sf_offsets(rows, d, operand):
    """Byte offset of the scale of (row r, 32-element block kb32) in sf_out -- include/sq_score.h, sq_score_quantize_mx."""
    G, P = (128, 1) if operand == 0 else (224, 2)
    ngroups = -(-rows // G)
    r = np.arange(rows)[:, None]
    kb32 = np.arange(-(-d // 32))[None, :]
    rg = r % G
    return ((kb32 // 4 * ngroups + r // G) * P + rg // 128) * 512 + (r % 32) * 16 + (rg // 32 % 4) * 4 + kb32 % 4


def check_quantised(q, sf, X, operand):
    rows, d = X.shape
    codes, exps = O.quantize_mx(X)
    off = sf_offsets(rows, d, operand)
    assert sf.shape[0] >= off.max() + 1
    got_e = sf[off].astype(np.int32) - 127
    np.testing.assert_array_equal(got_e, exps)
    table = O.e4m3_values()
    assert not np.isnan(table[q]).any()
    np.testing.assert_array_equal(table[q], table[codes])          # +0 and -0 are the same value
    rest = np.ones(sf.shape[0], dtype=bool)
    rest[off.ravel()] = False
    assert (sf[rest] == 0).all()                                   # bytes no row / block reaches


@pytest.mark.parametrize("operand", [0, 1], ids=["H", "W"])
@pytest.mark.parametrize("rows,d", [(5, 16), (33, 208), (300, 4096), (225, 2880), (1000, 5120), (129, 64), (449, 48)])
def test_quantize_mx_is_bit_exact(rows, d, operand):
    sq = _sq()
    gen = torch.Generator().manual_seed(rows * 7 + d)
    X = torch.randn(rows, d, generator=gen) * torch.exp(torch.rand(rows, 1, generator=gen) * 6 - 4)
    X = X * torch.exp(torch.randn(rows, d, generator=gen) * 2)    # a wide dynamic range inside every row
    X = X.to(torch.bfloat16)
    X[rows // 2] = 0                                               # an all-zero row
    X[0, 0] = 3.0e4                                                # an outlier: only its own block pays for it
    X[1, : min(d, 32)] = torch.tensor([448.0 * 2.0 ** (i % 5 - 2) for i in range(min(d, 32))]).to(torch.bfloat16)   # block maxima on 448 * 2^e
    X[2, : min(d, 16)] = torch.tensor([m / 16.0 + 1 / 32.0 for m in range(min(d, 16))]).to(torch.bfloat16)          # ties
    if rows > 4:
        X[3] = X[3] * 1e-30; X[4] = X[4] * 1e30                    # near the ends of the exponent range (incl. subnormal inputs)
        X[3, 0] = 1e-40
    eng = sq.SqScore(d, 1000, max_tokens=rows, max_seqs=1)
    q, sf = eng.quantize_mx(X.to(DEV), operand)
    torch.cuda.synchronize()
    check_quantised(q.cpu().numpy(), sf.cpu().numpy(), X, operand)
    eng.close()


def _run_mx(inp, k, window, **kw):
    sq = _sq()
    wl = inp["workload"]
    eng = sq.SqScore(wl.d, wl.V, max_tokens=inp["T"], max_seqs=inp["B"], max_k=k, **kw)
    Hq, hsf = eng.quantize_mx(inp["H"].to(DEV), sq.MX_OPERAND_H)
    Wq, wsf = eng.quantize_mx(inp["W"].to(DEV), sq.MX_OPERAND_W)
    out = eng.run_mx(Hq, hsf, Wq, wsf, inp["targets"].to(DEV), inp["cu_seqlens"].to(DEV), k, window)
    torch.cuda.synchronize()
    out2 = eng.run_mx(Hq, hsf, Wq, wsf, inp["targets"].to(DEV), inp["cu_seqlens"].to(DEV), k, window)   # deterministic
    torch.cuda.synchronize()
    for n in ("lse", "target_logprob", "entropy", "conf", "topk_logprob"):
        assert torch.equal(out[n], out2[n]), n
    eng.close()
    check_quantised(Hq.cpu().numpy(), hsf.cpu().numpy(), inp["H"], 0)
    check_quantised(Wq.cpu().numpy(), wsf.cpu().numpy(), inp["W"], 1)
    Hd = O.dequantize_mx(*O.quantize_mx(inp["H"]))
    Wd = O.dequantize_mx(*O.quantize_mx(inp["W"]))
    return {n: v.cpu().numpy() for n, v in out.items()}, Hd, Wd


@pytest.mark.parametrize("cg,chunks", [(2, 0), (1, 0), (2, 3)])
@pytest.mark.parametrize("d,V", [(64, 1024), (208, 1003), (4096, 600), (512, 224), (128, 449)])
def test_mx_scores_match_oracle_on_quantised_operands(d, V, cg, chunks):
    wl = workloads.custom(name="mx", d=d, V=V, B=3, len_lo=60, len_hi=200, k=5, window=16, seed=170 + d, w_std=0.05,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    out, Hd, Wd = _run_mx(inp, wl.k, wl.window, cta_group=cg, num_chunks=chunks)
    ref = O.score(Hd, Wd, inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
    check_tokens(out, ref, wl.k)
    check_seqs(out, ref)


def test_mx_rows_with_a_wide_dynamic_range():
    """Where block scaling differs from one scale per row: rows of H whose blocks span many binades."""
    wl = workloads.custom(name="mx_wide", d=256, V=700, B=2, len_lo=150, len_hi=300, k=8, window=8, seed=181, w_std=0.05,
                          planted_frac=0.3, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    g = torch.Generator().manual_seed(9)
    gain = torch.exp2(torch.randint(-12, 6, (1, wl.d // 32), generator=g).float()).repeat_interleave(32, dim=1)
    inp["H"] = (inp["H"].float() * gain).to(torch.bfloat16)
    inp["W"] = (inp["W"].float() / gain).to(torch.bfloat16)        # the logits keep their size, the operands do not
    out, Hd, Wd = _run_mx(inp, wl.k, wl.window)
    ref = O.score(Hd, Wd, inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
    check_tokens(out, ref, wl.k)
    check_seqs(out, ref)


def test_mx_decode_shaped():
    wl = workloads.custom(name="mx_dec", d=1024, V=40000, B=2, len_lo=20, len_hi=40, k=20, window=8, seed=183, w_std=0.03,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    out, Hd, Wd = _run_mx(inp, wl.k, wl.window)
    ref = O.score(Hd, Wd, inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
    check_tokens(out, ref, wl.k)
    check_seqs(out, ref)


def test_mx_model_shaped_sampled_rows_and_distance_to_bf16():
    sq = _sq()
    wl = workloads.custom(name="mx_model", d=4096, V=151936, B=4, len_lo=100, len_hi=250, k=20, window=64, seed=75,
                          w_std=0.02, planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    eng = sq.SqScore(wl.d, wl.V, max_tokens=inp["T"], max_seqs=inp["B"], max_k=wl.k)
    Hq, hsf = eng.quantize_mx(inp["H"].to(DEV), sq.MX_OPERAND_H)
    Wq, wsf = eng.quantize_mx(inp["W"].to(DEV), sq.MX_OPERAND_W)
    out = eng.run_mx(Hq, hsf, Wq, wsf, inp["targets"].to(DEV), inp["cu_seqlens"].to(DEV), wl.k, wl.window)
    torch.cuda.synchronize()
    out = {n: v.cpu().numpy() for n, v in out.items()}
    rows = np.unique(np.concatenate([[0, inp["T"] - 1], np.random.default_rng(4).integers(0, inp["T"], 20)]))
    # W: the GPU's codes and scales against the definition on a sample of rows, then the oracle's own dequantisation
    wrows = np.unique(np.concatenate([[0, 223, 224, wl.V - 1], np.random.default_rng(5).integers(0, wl.V, 400)]))
    codes_w, exps_w = O.quantize_mx(inp["W"])
    off = sf_offsets(wl.V, wl.d, 1)
    np.testing.assert_array_equal(wsf.cpu().numpy()[off[wrows]].astype(np.int32) - 127, exps_w[wrows])
    table = O.e4m3_values()
    np.testing.assert_array_equal(table[Wq.cpu().numpy()[wrows]], table[codes_w[wrows]])
    Wd = O.dequantize_mx(codes_w, exps_w)
    Hd = O.dequantize_mx(*O.quantize_mx(inp["H"][rows]))
    ref = O.token_scores(Hd, Wd, inp["targets"].numpy()[rows], wl.k)
    check_tokens(out, ref, wl.k, rows=rows)
    # what the quantisation costs against the bf16 path's own oracle, next to the per-tensor FP8 variant's
    ref16 = O.token_scores(inp["H"][rows], O.widen(inp["W"]), inp["targets"].numpy()[rows], wl.k)
    Hq8, hs8 = eng.quantize_fp8(inp["H"].to(DEV), False)
    Wq8, ws8 = eng.quantize_fp8(inp["W"].to(DEV), True)
    out8 = eng.run_fp8(Hq8, hs8, Wq8, ws8, inp["targets"].to(DEV), inp["cu_seqlens"].to(DEV), wl.k, wl.window)
    torch.cuda.synchronize()
    out8 = {n: v.cpu().numpy() for n, v in out8.items()}
    eng.close()
    err = {}
    for name, o in (("mx", out), ("fp8", out8)):
        err[name] = [np.abs(o[n][rows] - ref16[n]).max() for n in ("lse", "target_logprob", "conf")]
        print("%s vs bf16 oracle: max |d lse| %.4f  |d target_logprob| %.4f  |d conf| %.4f" % (name, *err[name]))
    assert err["mx"][0] < 0.05 and err["mx"][1] < 0.5 and err["mx"][2] < 0.2


def test_mx_rejects_bad_arguments():
    sq = _sq()
    eng = sq.SqScore(72, 512, max_tokens=32, max_seqs=2, max_k=5)      # d % 16 != 0
    X = torch.zeros(32, 72, dtype=torch.bfloat16, device=DEV)
    with pytest.raises(sq.SqScoreError) as ei:
        eng.quantize_mx(X, sq.MX_OPERAND_H)
    assert ei.value.code == sq.ERR_UNSUPPORTED
    eng.close()
    assert sq.lib().sq_score_mx_scale_bytes(300, 4096, 0) == 32 * 3 * 512
    assert sq.lib().sq_score_mx_scale_bytes(300, 4096, 1) == 32 * 2 * 1024
    assert sq.lib().sq_score_mx_scale_bytes(300, 4096, 2) == -1
