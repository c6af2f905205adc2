"""sq_score_reduce_static: kernel 2 for callers that cannot allocate device memory.

Who that is: a plug-in inside a serving engine that gave all free HBM to its own pool at start-up (a cudaMalloc made by
a library fails there, or takes memory the engine has budgeted), and code in a latency-critical loop, where cudaMalloc /
cudaFree may stall every stream of the process.  Such callers cannot create a ctx either (sq_score_create allocates the
workspace), so the entry point takes no ctx and keeps its scratch in a fixed array inside the library.

The checks: its results against the existing path's (SqScore.reduce on a ctx) at the tolerance of the parity tests, on
two calls in a row with different inputs -- the array keeps whatever the previous call left, so the second call is the
one that would show a stale counter or partial -- and once more after the array has been used by a call with other
sizes; sizes beyond the stated maximum are refused with a message; the device's free memory does not shrink across a
call.  This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It does not depend on them: the static call comes first, before any ctx exists in this test.
"""
import numpy as np
import pytest
import torch

import workloads

REL_TOL = 1e-3      # the sequence aggregates' tolerance in tests/test_parity_gpu.py (check_seqs)
ABS_TOL = 1e-6
SEQ_KEYS = ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")


def _inputs(num_seqs, len_lo, len_hi, seed, with_targets, dev):
    r = workloads.reduction_inputs(num_seqs, len_lo, len_hi, seed=seed)
    g = torch.Generator().manual_seed(seed + 1)
    tg = None
    if with_targets:
        tg = torch.randint(0, 1000, (r["T"],), generator=g, dtype=torch.int32)
        tg[torch.rand(r["T"], generator=g) < 0.2] = -1                      # "no target" tokens
    a = {n: r[n].to(dev) for n in ("target_logprob", "entropy", "conf", "cu_seqlens")}
    a["targets"] = None if tg is None else tg.to(dev)
    a["T"], a["B"] = r["T"], r["B"]
    return a


def _compare(got, want):
    for key in SEQ_KEYS:
        a, b = got[key].cpu().numpy(), want[key].cpu().numpy()
        assert (np.isnan(a) == np.isnan(b)).all(), key
        ok = ~np.isnan(b)
        np.testing.assert_allclose(a[ok], b[ok], rtol=REL_TOL, atol=ABS_TOL, err_msg=key)


@pytest.mark.gpu
def test_reduce_static_matches_the_ctx_path_on_two_calls_in_a_row():
    import paper_2604_07725_b200 as sq
    dev = torch.device("cuda:0")
    # call 1: many short sequences (empty ones among them), targets with invalid entries, a window inside the sequences
    # call 2: fewer, longer sequences spanning several 8192-token tiles, no targets, another window -- other tile and
    #         sequence counts than call 1, so anything call 1 left in the array would be in the way
    cases = [(_inputs(3000, 0, 700, 11, True, dev), 256), (_inputs(40, 1, 30000, 12, False, dev), 2048)]
    outs = []
    for a, window in cases:                                     # the static path first: no ctx exists yet
        out = {n: torch.full((a["B"],), -7.0, dtype=torch.float32, device=dev) for n in SEQ_KEYS}   # caller-owned
        got = sq.reduce_static(a["target_logprob"], a["entropy"], a["conf"], a["cu_seqlens"], window,
                               targets=a["targets"], vocab=1000, out=out)
        assert got is out
        outs.append(out)
    torch.cuda.synchronize()
    for (a, window), got in zip(cases, outs):                   # the existing path: a ctx with its own workspace
        eng = sq.SqScore(64, 1000, max_tokens=a["T"], max_seqs=a["B"], max_k=5, reduce_only=True)
        want = eng.reduce(a["target_logprob"], a["entropy"], a["conf"], a["cu_seqlens"], window, targets=a["targets"])
        torch.cuda.synchronize()
        _compare(got, want)
        eng.close()
    # back to the first input after the array served the second, with the free memory watched across the call
    a, window = cases[0]
    eng = sq.SqScore(64, 1000, max_tokens=a["T"], max_seqs=a["B"], max_k=5, reduce_only=True)
    want = eng.reduce(a["target_logprob"], a["entropy"], a["conf"], a["cu_seqlens"], window, targets=a["targets"])
    out = {n: torch.empty(a["B"], dtype=torch.float32, device=dev) for n in SEQ_KEYS}
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(dev)[0]
    sq.reduce_static(a["target_logprob"], a["entropy"], a["conf"], a["cu_seqlens"], window, targets=a["targets"],
                     vocab=1000, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(dev)[0] >= free_before, "the call took device memory"
    _compare(out, want)
    eng.close()


@pytest.mark.gpu
def test_reduce_static_refuses_sizes_beyond_its_fixed_scratch():
    import paper_2604_07725_b200 as sq
    dev = torch.device("cuda:0")
    one = torch.zeros(8, dtype=torch.float32, device=dev)
    cu_many = torch.zeros(sq.STATIC_MAX_SEQS + 2, dtype=torch.int32, device=dev)       # B = maximum + 1
    with pytest.raises(sq.SqScoreError) as e:
        sq.reduce_static(one, one, one, cu_many, 4)
    assert e.value.code == sq.ERR_INVALID_ARG and "at most" in str(e.value) and str(sq.STATIC_MAX_SEQS) in str(e.value)
    # T = maximum + 1: only the size is looked at before the refusal, so a small tensor stands in for the arrays
    L = sq.lib()
    out = torch.zeros(1, dtype=torch.float32, device=dev)
    cu = torch.tensor([0, sq.STATIC_MAX_TOKENS + 1], dtype=torch.int32, device=dev)
    rc = L.sq_score_reduce_static(one.data_ptr(), one.data_ptr(), one.data_ptr(), None, cu.data_ptr(),
                                  sq.STATIC_MAX_TOKENS + 1, 1, 1, 4, out.data_ptr(), out.data_ptr(), out.data_ptr(),
                                  out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert rc == sq.ERR_INVALID_ARG and b"at most" in L.sq_score_last_error(None)
    torch.cuda.synchronize()
    assert float(out[0]) == 0.0                                   # nothing was launched
    # the maximum number of sequences itself is served (all but one empty -> NaNs there)
    cu_max = torch.zeros(sq.STATIC_MAX_SEQS + 1, dtype=torch.int32, device=dev)
    cu_max[-1] = 8
    got = sq.reduce_static(one, one, one + 2.0, cu_max, 4)
    torch.cuda.synchronize()
    assert torch.isnan(got["seq_mean_conf"][:-1]).all() and float(got["seq_mean_conf"][-1]) == 2.0
    assert float(got["seq_min_window_conf"][-1]) == 2.0 and float(got["seq_mean_logprob"][-1]) == 0.0
