"""Memory-safety checks of the CUDA path that need no external tool (compute-sanitizer is closed on this GPU pool, so
memcheck / initcheck cannot be run there):

  * guard bands: every caller-owned buffer (inputs and outputs) sits between two guard regions filled with a
    pattern; after the run the guards must be intact (no out-of-bounds WRITE on a caller buffer) and every output
    word must have been overwritten (outputs are pre-filled with a signalling pattern);
  * workspace poisoning: sq_score_debug_fill_workspace fills every ctx-owned workspace and staging buffer with 0xFF
    bytes (NaN floats, -1 ints) before the run; the results must be bit-identical to a run on a fresh ctx and match
    the oracle, so no kernel reads workspace it did not write in the same run (what initcheck would report);
  * repeated runs on one ctx with different shapes (stale partial states from a larger run must never leak into a
    smaller one).
Cases: tiny, ragged multi-chunk, decode-shaped (148 chunks), host-streaming form, shard + merge, FP8, prepare / run_x,
kernel 2 alone with arrays whose length is not a multiple of 4."""
import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O
from test_parity_gpu import SEQ_KEYS, check_seqs, check_tokens

pytestmark = pytest.mark.gpu
DEV = torch.device("cuda:0")
GUARD = 4096            # bytes on each side
PATTERN = 0xA5


def _sq():
    import paper_2604_07725_b200 as sq
    return sq


class Guarded:
    """A device tensor of the given shape/dtype placed between two guard bands inside one allocation."""

    def __init__(self, shape, dtype, fill_from=None, prefill=None):
        n = int(np.prod(shape)) * torch.empty(0, dtype=dtype).element_size()
        pad = (-n) % 16
        self.raw = torch.full((GUARD + n + pad + GUARD,), PATTERN, dtype=torch.uint8, device=DEV)
        self.n, self.pad = n, pad
        self.t = self.raw[GUARD:GUARD + n].view(dtype).view(*shape)
        if fill_from is not None:
            self.t.copy_(fill_from.to(DEV))
        elif prefill is not None:
            self.raw[GUARD:GUARD + n] = prefill

    def guards_intact(self):
        lo = self.raw[:GUARD]
        hi = self.raw[GUARD + self.n:]
        return bool((lo == PATTERN).all()) and bool((hi == PATTERN).all())

    def fully_written(self, prefill):
        """No 4-byte word of the payload still holds the prefill pattern."""
        w = self.raw[GUARD:GUARD + self.n].view(torch.int32)
        pat = int.from_bytes(bytes([prefill] * 4), "little", signed=True)
        return not bool((w == pat).any())


def guarded_outputs(T, B, k):
    shapes = {"lse": ((T,), torch.float32), "target_logprob": ((T,), torch.float32), "entropy": ((T,), torch.float32),
              "conf": ((T,), torch.float32), "topk_logprob": ((T, k), torch.float32), "topk_index": ((T, k), torch.int32)}
    shapes.update({n: ((B,), torch.float32) for n in SEQ_KEYS})
    return {n: Guarded(s, dt, prefill=0xEE) for n, (s, dt) in shapes.items()}


def check_guards(bufs, written=True):
    for n, g in bufs.items():
        assert g.guards_intact(), "out-of-bounds write next to %s" % n
        if written and g.n:
            assert g.fully_written(0xEE), "%s was not fully written" % n


CASES = [
    dict(name="tiny", wl=dict(d=64, V=1024, B=4, len_lo=32, len_hi=96, k=5, window=16, seed=1001, w_std=0.05), eng={}),
    dict(name="ragged_chunks", wl=dict(d=200, V=1003, B=3, len_lo=100, len_hi=300, k=20, window=16, seed=5, w_std=0.1), eng=dict(num_chunks=3, group_m=2)),
    dict(name="single_cta", wl=dict(d=72, V=2500, B=2, len_lo=50, len_hi=130, k=8, window=8, seed=6, w_std=0.1), eng=dict(cta_group=1)),
    dict(name="decode", wl=dict(d=128, V=40000, B=1, len_lo=7, len_hi=7, k=20, window=4, seed=57, w_std=0.1), eng={}),
]


@pytest.mark.parametrize("case", CASES, ids=[c["name"] for c in CASES])
def test_guard_bands_and_poisoned_workspace(case):
    sq = _sq()
    wl = workloads.custom(name=case["name"], **case["wl"])
    inp = workloads.make_inputs(wl)
    T, B, k = inp["T"], inp["B"], wl.k
    ins = {"H": Guarded((T, wl.d), torch.bfloat16, inp["H"]), "W": Guarded((wl.V, wl.d), torch.bfloat16, inp["W"]),
           "targets": Guarded((T,), torch.int32, inp["targets"]), "cu": Guarded((B + 1,), torch.int32, inp["cu_seqlens"])}
    ref = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], k, wl.window)
    eng = sq.SqScore(wl.d, wl.V, max_tokens=T + 300, max_seqs=B + 3, max_k=k, **case["eng"])
    # (1) a larger, unrelated run first: its partial states stay behind in the workspace
    big = workloads.make_inputs(workloads.custom(name="stale", d=wl.d, V=wl.V, B=B + 3, len_lo=(T + 300) // (B + 3), len_hi=(T + 300) // (B + 3),
                                                 k=k, window=3, seed=99, w_std=1.0))
    eng.run(big["H"].to(DEV), big["W"].to(DEV), big["targets"].to(DEV), big["cu_seqlens"].to(DEV), k, 3)
    outs = guarded_outputs(T, B, k)
    o1 = eng.run(ins["H"].t, ins["W"].t, ins["targets"].t, ins["cu"].t, k, wl.window, out={n: g.t for n, g in outs.items()})
    torch.cuda.synchronize()
    check_guards(outs); check_guards(ins, written=False)
    first = {n: v.clone() for n, v in o1.items()}
    # (2) the same run on a poisoned workspace: bit-identical, and equal to the oracle
    eng.debug_fill_workspace(0xFF)
    outs2 = guarded_outputs(T, B, k)
    o2 = eng.run(ins["H"].t, ins["W"].t, ins["targets"].t, ins["cu"].t, k, wl.window, out={n: g.t for n, g in outs2.items()})
    torch.cuda.synchronize()
    check_guards(outs2); check_guards(ins, written=False)
    for n in first:
        assert torch.equal(first[n], o2[n]) or (torch.isnan(first[n]) == torch.isnan(o2[n])).all(), n
    got = {n: v.cpu().numpy() for n, v in o2.items()}
    check_tokens(got, ref, k)
    check_seqs(got, ref)
    eng.close()


def test_host_form_shard_merge_fp8_and_run_x_on_poisoned_workspace():
    sq = _sq()
    wl = workloads.custom(name="forms", d=256, V=3000, B=3, len_lo=100, len_hi=400, k=20, window=32, seed=41, w_std=0.1,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    T, B, k = inp["T"], inp["B"], wl.k
    H, W, tg, cu = (inp[n].to(DEV) for n in ("H", "W", "targets", "cu_seqlens"))
    ref = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], k, wl.window)
    eng = sq.SqScore(wl.d, wl.V, max_tokens=T + 64, max_seqs=B, max_k=k, staging=True)
    # host-streaming form
    eng.debug_fill_workspace(0xFF)
    host = torch.full((4 * B,), float("nan")).pin_memory()
    eng.run_host(inp["H"].pin_memory(), W, inp["targets"].pin_memory(), inp["cu_seqlens"].pin_memory(), k, wl.window, host)
    torch.cuda.synchronize()
    check_seqs({n: host[i * B:(i + 1) * B].numpy() for i, n in enumerate(SEQ_KEYS)}, ref)
    # shard + merge with guarded state buffers (three uneven shards, one ctx)
    eng.debug_fill_workspace(0xFF)
    starts = [0, 1024, 1100, 3000]
    words = sq.shard_state_bytes(T, k) // 4
    states = Guarded((3, words), torch.float32, prefill=0xEE)
    for r in range(3):
        eng.run_shard(H, W[starts[r]:starts[r + 1]], starts[r], tg, k, out=states.t[r])
    torch.cuda.synchronize()
    assert states.guards_intact() and states.fully_written(0xEE)
    eng.debug_fill_workspace(0xFF)
    outs = guarded_outputs(T, B, k)
    om = eng.merge_shards(states.t, starts, tg, cu, k, wl.window, out={n: g.t for n, g in outs.items()})
    torch.cuda.synchronize()
    check_guards(outs)
    got = {n: v.cpu().numpy() for n, v in om.items()}
    check_tokens(got, ref, k); check_seqs(got, ref)
    # FP8 variant: guarded codes and scales, poisoned workspace
    eng.debug_fill_workspace(0xFF)
    q = Guarded((T, wl.d), torch.uint8, prefill=0xEE); sc = Guarded((T,), torch.float32, prefill=0xEE)
    Hq, hs = eng.quantize_fp8(H, False, out=(q.t, sc.t))
    Wq, ws = eng.quantize_fp8(W, True)
    o8 = eng.run_fp8(Hq, hs, Wq, ws, tg, cu, k, wl.window)
    torch.cuda.synchronize()
    assert q.guards_intact() and sc.guards_intact() and sc.fully_written(0xEE)
    ref8 = O.score(O.dequantize_fp8(Hq.cpu().numpy(), hs.cpu().numpy()), O.dequantize_fp8(Wq.cpu().numpy(), ws.cpu().numpy()),
                   inp["targets"], inp["cu_seqlens"], k, wl.window)
    g8 = {n: v.cpu().numpy() for n, v in o8.items()}
    check_tokens(g8, ref8, k); check_seqs(g8, ref8)
    # prepare / run_x with a guarded H output
    pre = workloads.prepare_inputs(wl, query_lo=1, query_hi=30)
    pos, pcu = O.trajectory_positions(pre["query_lens"], pre["traj_lens"])
    eng.debug_fill_workspace(0xFF)
    Hout = Guarded((pre["T"], wl.d), torch.bfloat16, prefill=0xEE)
    pd, cd = eng.positions(pre["query_lens"].to(torch.int32).to(DEV), pre["traj_lens"].to(torch.int32).to(DEV), pre["T"])
    eng.prepare(pre["X"].to(DEV), pd, pre["gain"].to(DEV), pre["eps"], out=Hout.t)
    ox = eng.run_x(pre["X"].to(DEV), pd, pre["gain"].to(DEV), pre["eps"], W, pre["targets"].to(DEV), cd, k, wl.window)
    torch.cuda.synchronize()
    assert Hout.guards_intact()
    refx = O.score(O.round_to_bf16(O.prepare_hidden(pre["X"], pos, pre["gain"], pre["eps"])), inp["W"], pre["targets"], pcu, k, wl.window)
    gx = {n: v.cpu().numpy() for n, v in ox.items()}
    check_tokens(gx, refx, k); check_seqs(gx, refx)
    eng.close()


@pytest.mark.parametrize("window", [1, 5, 2048, 8193])
@pytest.mark.parametrize("dbg", [None, "256"], ids=["default", "streaming"])
def test_reduce_alone_guarded_arrays_and_poisoned_workspace(window, dbg):
    """Kernel 2 reads ahead of the current token (window look-ahead, 16-byte vectors): the per-token arrays end exactly
    where their guard band begins and have a length that is not a multiple of 4."""
    sq = _sq()
    lens = [3, 8190, 1, 0, 8193, 12289, 2, 4095]
    T = sum(lens)
    g = torch.Generator().manual_seed(5)
    lp = -(torch.rand(T, generator=g) * 12); en = torch.rand(T, generator=g) * 11; cf = 3 + torch.rand(T, generator=g) * 12
    cu = torch.tensor(np.concatenate([[0], np.cumsum(lens)]), dtype=torch.int32)
    ref = O.sequence_scores(lp.numpy(), en.numpy(), cf.numpy(), cu.numpy(), window)
    G = {n: Guarded((T,), torch.float32, v) for n, v in (("lp", lp), ("en", en), ("cf", cf))}
    # NaN guards right behind the arrays: a read past the end would poison the window sums
    for gd in G.values():
        gd.raw[GUARD + gd.n:].view(torch.float32)[:] = float("nan")
    import os
    eng = sq.SqScore(64, 1000, max_tokens=T, max_seqs=len(lens), max_k=5, reduce_only=True, debug_flags=int(dbg or 0))
    eng.debug_fill_workspace(0xFF)
    out = eng.reduce(G["lp"].t, G["en"].t, G["cf"].t, cu.to(DEV), window)
    torch.cuda.synchronize()
    check_seqs({n: v.cpu().numpy() for n, v in out.items()}, ref)
    eng.close()
