"""The N > 1 entry points on the real NCCL backend, at the one world size this box allows (1 rank, 1 GPU): the
data-parallel step's exchange (sharding.gather_sequence_scores: one all_gather_into_tensor, scatter by id on the
device) and the whole vocab-parallel step (sharding.score_vocab_parallel: shard kernels -> all-gather of the packed
state on the compute stream -> merge), both against the fp64 oracle.  Multi-rank layouts are covered with gloo on CPU
(tests/test_sharding_gloo.py) and every shard count on one GPU in tests/test_vocab_parallel_gpu.py."""
import os
import socket

import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O
from test_parity_gpu import check_seqs, check_tokens

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def test_nccl_world_size_one_runs_both_exchanges():
    import torch.distributed as dist
    import paper_2604_07725_b200 as sq
    from paper_2604_07725_b200 import sharding
    dev = torch.device("cuda:0")
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(_free_port())
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    try:
        wl = workloads.custom(name="nccl1", d=128, V=2100, B=5, len_lo=30, len_hi=200, k=20, window=16, seed=66, w_std=0.2,
                              planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
        inp = workloads.make_inputs(wl, lengths=[40, 0, 150, 7, 90])
        ref = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
        H, W, tg, cu = (inp[n].to(dev) for n in ("H", "W", "targets", "cu_seqlens"))
        eng = sq.SqScore(wl.d, wl.V, max_tokens=inp["T"], max_seqs=inp["B"], max_k=wl.k)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            # data-parallel: this rank owns sequences in a permuted order; the gather puts them back by id
            ids, local_cu, rows = sharding.local_batch(inp["cu_seqlens"], 0, 1)
            out = eng.run(H, W, tg, cu, wl.k, wl.window, stream=st)
            perm = [3, 0, 4, 1, 2]
            local = {n: out[n][perm] for n in sharding.SEQ_KEYS}
            got = sharding.gather_sequence_scores(local, perm, inp["B"], 1, device=dev)
            # vocab-parallel with one rank that owns every row
            out_v = sharding.score_vocab_parallel(eng, H, W, [0, wl.V], 0, tg, cu, wl.k, wl.window, stream=st)
            # the same with the states read in place: ready() / release() are 4-byte NCCL all-reduces on this stream
            state = torch.empty(sq.shard_state_bytes(inp["T"], wl.k) // 4, dtype=torch.float32, device=dev)
            peers = sharding.PeerStates(state, 0, 1)
            out_p = sharding.score_vocab_parallel_peer(eng, peers, H, W, [0, wl.V], tg, cu, wl.k, wl.window, stream=st)
        st.synchronize()
        # a stream that is NOT the current one: what the step allocates (packed state, gathered states, outputs) must still
        # belong to that stream -- default-stream tensors allocated right behind the call must not land on its blocks
        st2 = torch.cuda.Stream()
        st2.wait_stream(torch.cuda.current_stream())
        assert torch.cuda.current_stream() != st2
        out_s = sharding.score_vocab_parallel(eng, H, W, [0, wl.V], 0, tg, cu, wl.k, wl.window, stream=st2)
        junk = [torch.full((sq.shard_state_bytes(inp["T"], wl.k) // 4,), float("nan"), device=dev) for _ in range(8)]
        st2.synchronize()
        torch.cuda.synchronize()
        del junk
        for n in ("lse", "conf", "topk_index", "seq_min_window_conf"):
            assert torch.equal(torch.nan_to_num(out_s[n].float(), nan=-7.0), torch.nan_to_num(out_v[n].float(), nan=-7.0)), n
        for n in ("lse", "conf", "topk_index", "seq_min_window_conf"):             # (the empty sequence's NaN equals itself here)
            assert torch.equal(torch.nan_to_num(out_p[n].float(), nan=-7.0), torch.nan_to_num(out_v[n].float(), nan=-7.0)), n
        assert got["seq_mean_conf"].is_cuda
        check_seqs({n: v.cpu().numpy() for n, v in got.items()}, ref)
        o = {n: v.cpu().numpy() for n, v in out_v.items()}
        check_tokens(o, ref, wl.k)
        check_seqs(o, ref)
        for n in ("lse", "conf", "topk_index"):                       # and identical to the single-GPU path
            assert torch.equal(out_v[n], out[n]), n
        eng.close()
    finally:
        dist.destroy_process_group()
