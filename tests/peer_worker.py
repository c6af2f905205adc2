"""Worker of tests/test_vocab_parallel_gpu.py::test_peer_exchange_two_processes_on_one_gpu (launched by torchrun, one
process per rank, both on cuda:0): vocab-parallel scoring with the peers' states read in place."""
import os

import numpy as np
import torch
import torch.distributed as dist

import workloads
from oracle import sq_oracle as O
from test_parity_gpu import check_seqs, check_tokens


def main():
    import paper_2604_07725_b200 as sq
    from paper_2604_07725_b200 import sharding
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    wl = workloads.custom(name="peer", d=200, V=1003, B=3, len_lo=40, len_hi=200, k=20, window=16, seed=62, w_std=0.2,
                          planted_frac=0.5, planted_scale=3.0, rmsnorm=True)
    inp = workloads.make_inputs(wl)
    starts = [0, 620, 1003]                                  # uneven, not tile-aligned
    T, B = inp["T"], inp["B"]
    eng = sq.SqScore(wl.d, 620, max_tokens=T, max_seqs=B, max_k=wl.k)
    H = inp["H"].to(dev); W = inp["W"].to(dev); tg = inp["targets"].to(dev); cu = inp["cu_seqlens"].to(dev)
    state = torch.empty(sq.shard_state_bytes(T, wl.k) // 4, dtype=torch.float32, device=dev)
    peers = sharding.PeerStates(state, rank, world)
    ref = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], wl.k, wl.window)
    for step in range(3):                                    # the buffers are reused: ready / release order the steps
        out = sharding.score_vocab_parallel_peer(eng, peers, H, W[starts[rank]:starts[rank + 1]], starts, tg, cu, wl.k, wl.window)
        torch.cuda.synchronize()
        o = {n: v.cpu().numpy() for n, v in out.items()}
        check_tokens(o, ref, wl.k)
        check_seqs(o, ref)
    dist.barrier()
    eng.close()
    print("peer exchange OK rank %d" % rank, flush=True)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
