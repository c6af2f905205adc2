"""GPU parity of vocab-parallel scoring: the LM head split by rows over R shards, one packed
partial state per shard, merged by the associative operator -- against the fp64 oracle on the WHOLE vocabulary, and
against the single-shard GPU path.  The shards run one after another on one GPU (nothing waits on anything), exactly
the kernels each rank of a tensor-parallel scorer would run; the exchange itself is covered on CPU with gloo."""
import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O
from test_parity_gpu import check_seqs, check_tokens, run_gpu

pytestmark = pytest.mark.gpu
DEV = torch.device("cuda:0")


def _sq():
    import paper_2604_07725_b200 as sq
    return sq


def run_sharded(inp, starts, k, window, targets=None):
    """Every shard through ONE ctx sized for the largest shard (the layout sharding.score_vocab_parallel uses: uneven
    shards pass their own row count to sq_score_run_shard)."""
    sq = _sq()
    wl = inp["workload"]
    T, B = inp["T"], inp["B"]
    H = inp["H"].to(DEV); W = inp["W"].to(DEV); cu = inp["cu_seqlens"].to(DEV)
    tg = (inp["targets"] if targets is None else targets).to(DEV)
    eng = sq.SqScore(wl.d, max(1, max(starts[r + 1] - starts[r] for r in range(len(starts) - 1))), max_tokens=T, max_seqs=B, max_k=k)
    states = []
    for r in range(len(starts) - 1):
        v0, v1 = starts[r], starts[r + 1]
        if v1 == v0:
            states.append(eng.neutral_shard_state(T, k, device=DEV))
        else:
            states.append(eng.run_shard(H, W[v0:v1], v0, tg, k))          # a view into W: rows beyond v1 belong to the next shard
    allst = torch.stack(states)                       # what all_gather_into_tensor would return
    out = eng.merge_shards(allst, starts, tg, cu, k, window)
    # the same merge reading every state where it lies (sq_score_merge_shards_peer): separate allocations in no particular
    # address order -- what the peers' buffers are to the merge kernel -- must give the same bits
    pad = [torch.empty(1000 * (r + 1), device=DEV) for r in range(len(states))]
    scattered = [st.clone() for st in reversed(states)][::-1]
    outp = eng.merge_shards_peer(scattered, starts, tg, cu, k, window)
    torch.cuda.synchronize()
    for n in out:
        a, b = out[n], outp[n]
        assert torch.equal(a, b) or torch.equal(torch.isnan(a), torch.isnan(b)) and torch.equal(a[~torch.isnan(a)], b[~torch.isnan(b)]), n
    del pad
    eng.close()
    return {n: v.cpu().numpy() for n, v in out.items()}


@pytest.mark.parametrize("starts", [None, [0, 1003], [0, 100, 777, 1003], [0, 256, 256, 512, 1003], [0, 37, 74, 111, 500, 1003]],
                         ids=["tiles3", "one", "uneven3", "empty_shard", "five"])
def test_sharded_matches_oracle_and_single_gpu(starts):
    sq = _sq()
    wl = workloads.custom(name="vp", d=200, V=1003, B=3, len_lo=40, len_hi=200, k=20, window=16, seed=61, w_std=0.2,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    if starts is None:
        starts = sq.shard_vocab(wl.V, 3)
    tg = inp["targets"].clone()
    tg[0] = 0; tg[1] = wl.V - 1; tg[2] = -1; tg[3] = wl.V + 5      # edges of the vocabulary, invalid targets
    for i, v in enumerate(starts[1:-1]):                            # both sides of every shard boundary
        tg[4 + 2 * i] = max(0, v - 1); tg[5 + 2 * i] = min(wl.V - 1, v)
    out = run_sharded(inp, starts, wl.k, wl.window, targets=tg)
    ref = O.score(inp["H"], inp["W"], tg, inp["cu_seqlens"], wl.k, wl.window)
    check_tokens(out, ref, wl.k)
    check_seqs(out, ref)
    one = run_gpu(inp, targets=tg)
    for key in ("lse", "target_logprob", "entropy", "conf", "topk_logprob"):
        np.testing.assert_allclose(out[key], one[key], rtol=2e-5, atol=2e-5, err_msg=key)


def test_sharded_peaked_rows_keep_entropy_precision():
    """A strong planted peak (entropy ~1e-4 nats): the merged sums must keep the fp64 precision of S - 1 across the
    exchange (value + residue), or the rel-1e-3 bound on entropy fails."""
    wl = workloads.custom(name="vp_peak", d=128, V=3000, B=2, len_lo=50, len_hi=120, k=5, window=8, seed=62, w_std=0.1,
                          planted_frac=0.7, planted_scale=30.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    out = run_sharded(inp, [0, 1024, 2048, 3000], wl.k, wl.window)
    ref = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
    check_tokens(out, ref, wl.k)
    check_seqs(out, ref)


def test_sharded_model_shaped():
    """d = 2560, V = 151 936 over 8 shards (the tensor-parallel layout of a served scorer), 700 tokens; oracle on a row
    sample, the single-shard GPU path on all rows."""
    sq = _sq()
    wl = workloads.custom(name="vp_model", d=2560, V=151936, B=4, len_lo=100, len_hi=250, k=20, window=64, seed=63,
                          w_std=0.02, planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    starts = sq.shard_vocab(wl.V, 8)
    out = run_sharded(inp, starts, wl.k, wl.window)
    one = run_gpu(inp)
    for key in ("lse", "target_logprob", "entropy", "conf", "topk_logprob", "seq_mean_conf", "seq_min_window_conf"):
        np.testing.assert_allclose(out[key], one[key], rtol=2e-5, atol=2e-5, err_msg=key)
    rows = np.unique(np.concatenate([[0, inp["T"] - 1], np.random.default_rng(3).integers(0, inp["T"], 24)]))
    ref = O.token_scores(inp["H"][rows], O.widen(inp["W"]), inp["targets"].numpy()[rows], wl.k)
    check_tokens(out, ref, wl.k, rows=rows)


def test_score_vocab_parallel_entry_point_single_process():
    """sharding.score_vocab_parallel itself (the shipped entry point) with uneven shards and a ctx sized for the largest:
    one process plays every rank in turn with the collective replaced by a local stand-in that returns the stacked
    states (the NCCL form is exercised at world_size 1 in test_nccl_world1_gpu.py, the layout with gloo on CPU)."""
    sq = _sq()
    from paper_2604_07725_b200 import sharding
    wl = workloads.custom(name="vp_entry", d=128, V=1900, B=3, len_lo=40, len_hi=160, k=20, window=16, seed=64, w_std=0.2,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    starts = [0, 512, 1280, 1280, 1900]                                     # 512 / 768 / 0 / 620 rows
    H = inp["H"].to(DEV); W = inp["W"].to(DEV); cu = inp["cu_seqlens"].to(DEV); tg = inp["targets"].to(DEV)
    eng = sq.SqScore(wl.d, 768, max_tokens=inp["T"], max_seqs=inp["B"], max_k=wl.k)
    states = [None] * 4
    real_gather = sharding.gather_shard_states
    try:
        for phase in (0, 1):                                                # phase 0 collects every rank's state, phase 1 merges
            for r in range(4):
                def fake_gather(state, world, group=None, stream=None, r=r):
                    states[r] = state
                    return torch.stack([s if s is not None else torch.zeros_like(state) for s in states])
                sharding.gather_shard_states = fake_gather
                out = sharding.score_vocab_parallel(eng, H, W[starts[r]:starts[r + 1]], starts, r, tg, cu, wl.k, wl.window)
    finally:
        sharding.gather_shard_states = real_gather
    torch.cuda.synchronize()
    ref = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
    o = {n: v.cpu().numpy() for n, v in out.items()}
    check_tokens(o, ref, wl.k)
    check_seqs(o, ref)
    with pytest.raises(ValueError):
        sharding.score_vocab_parallel(eng, H, W[0:100], starts, 0, tg, cu, wl.k, wl.window)
    eng.close()


def test_shard_api_errors():
    sq = _sq()
    eng = sq.SqScore(64, 512, max_tokens=32, max_seqs=2, max_k=5)
    st = torch.zeros(2, sq.shard_state_bytes(32, 5) // 4, device=DEV)
    tg = torch.zeros(32, dtype=torch.int32, device=DEV); cu = torch.tensor([0, 16, 32], dtype=torch.int32, device=DEV)
    with pytest.raises(sq.SqScoreError):
        eng.merge_shards(st, [0, 600, 512], tg, cu, 5, 4)           # starts not monotone
    with pytest.raises(sq.SqScoreError):
        eng.merge_shards(st, [0, 512, 1024], tg, cu, 6, 4)          # k > max_k
    with pytest.raises(sq.SqScoreError):
        eng.run_shard(torch.zeros(32, 64, dtype=torch.bfloat16, device=DEV), torch.zeros(512, 64, dtype=torch.bfloat16, device=DEV), -1, tg, 5)
    with pytest.raises(sq.SqScoreError):             # more rows than the ctx was sized for
        eng.run_shard(torch.zeros(32, 64, dtype=torch.bfloat16, device=DEV), torch.zeros(513, 64, dtype=torch.bfloat16, device=DEV), 0, tg, 5)
    with pytest.raises(sq.SqScoreError):             # k larger than the shard
        eng.run_shard(torch.zeros(32, 64, dtype=torch.bfloat16, device=DEV), torch.zeros(3, 64, dtype=torch.bfloat16, device=DEV), 0, tg, 5)
    assert sq.shard_state_bytes(32, 5) == (6 + 2 * 8) * 32 * 4 and sq.shard_state_bytes(10, 20) == (6 + 40) * 40
    eng.close()


def test_peer_exchange_two_processes_on_one_gpu(tmp_path):
    """sharding.PeerStates + score_vocab_parallel_peer end to end: two processes (gloo for the host-side meeting points)
    open each other's state buffer through CUDA IPC and every one merges both states in place; each checks its result
    against the fp64 oracle.  On one GPU the peer's buffer is local memory -- the code path (handles, views, the pointer
    table of sq_score_merge_shards_peer, ready / release) is the one a multi-GPU node runs; no kernel waits on another."""
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", PYTHONPATH=root + os.pathsep + os.path.join(root, "tests"))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29731", os.path.join(root, "tests", "peer_worker.py")]
    res = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600, cwd=root)
    assert res.returncode == 0, res.stdout[-3000:] + res.stderr[-3000:]
    assert res.stdout.count("peer exchange OK") == 2, res.stdout[-2000:]
