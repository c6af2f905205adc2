"""world_size-2 gloo test (CPU) of the N>1 path's host logic: sequences are dealt to ranks, each
rank scores its own packed sub-batch (here with the fp64 oracle standing in for the kernels -- the
GPU is not available), and the all_gather puts the per-sequence scalars back in global order."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads
from oracle import sq_oracle as O
from paper_2604_07725_b200 import sharding


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.set_num_threads(1)
    wl = workloads.custom(name="shard", d=16, V=50, B=5, k=3, window=4, seed=17, w_std=0.5)
    inp = workloads.make_inputs(wl, lengths=[9, 0, 30, 4, 17])
    ids, local_cu, rows = sharding.local_batch(inp["cu_seqlens"], rank, world)
    tok = O.score(inp["H"][rows], inp["W"], inp["targets"][rows].numpy(), local_cu.numpy(), wl.k, wl.window)
    local = {k: torch.tensor(tok[k], dtype=torch.float32) for k in sharding.SEQ_KEYS}
    out = sharding.gather_sequence_scores(local, ids, inp["B"], world)
    if rank == 0:
        ret.update({k: v.numpy() for k, v in out.items()})
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_matches_single_rank():
    world = 2
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), ret), nprocs=world, join=True)
        got = dict(ret)
    wl = workloads.custom(name="shard", d=16, V=50, B=5, k=3, window=4, seed=17, w_std=0.5)
    inp = workloads.make_inputs(wl, lengths=[9, 0, 30, 4, 17])
    ref = O.score(inp["H"], inp["W"], inp["targets"].numpy(), inp["cu_seqlens"].numpy(), wl.k, wl.window)
    for key in sharding.SEQ_KEYS:
        a, b = got[key], ref[key]
        assert (np.isnan(a) == np.isnan(b)).all()
        np.testing.assert_allclose(a[~np.isnan(b)], b[~np.isnan(b)], rtol=1e-6)


def _few_worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ids = [0] if rank == 1 else []                      # more ranks than sequences: ranks 0 and 2 own nothing
    local = {k: torch.tensor([float(i + 1)]) if ids else torch.zeros(0) for i, k in enumerate(sharding.SEQ_KEYS)}
    out = sharding.gather_sequence_scores(local, ids, 1, world, device="cpu")
    ret[rank] = {k: v.clone() for k, v in out.items()}
    dist.barrier()
    dist.destroy_process_group()


def test_gather_with_ranks_that_own_no_sequence():
    """world > B: a rank without sequences still takes part in the ONE collective, on the collective's device."""
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_few_worker, args=(3, _free_port(), ret), nprocs=3, join=True)
        got = dict(ret)
    for r in range(3):
        for i, k in enumerate(sharding.SEQ_KEYS):
            assert got[r][k].tolist() == [float(i + 1)]


def test_local_batch_partitions_rows():
    cu = torch.tensor([0, 9, 9, 39, 43, 60], dtype=torch.int32)
    seen = []
    for r in range(3):
        ids, lcu, rows = sharding.local_batch(cu, r, 3)
        assert int(lcu[-1]) == len(rows)
        seen += rows.tolist()
        for i, b in enumerate(ids):
            assert int(lcu[i + 1] - lcu[i]) == int(cu[b + 1] - cu[b])
    assert sorted(seen) == list(range(60))


# ---------------------------------------------------------------------------------- vocab-parallel exchange (8(f)-4)
def test_shard_vocab_partition():
    import paper_2604_07725_b200 as sq
    for V, R in [(151936, 8), (201088, 4), (1003, 3), (100, 4), (256, 1), (257, 2)]:
        st = sq.shard_vocab(V, R)
        assert len(st) == R + 1 and st[0] == 0 and st[-1] == V and all(a <= b for a, b in zip(st, st[1:]))
        assert all(s % 256 == 0 for s in st[:-1])                       # shards start on vocab-tile boundaries
        sizes = [b - a for a, b in zip(st, st[1:])]
        assert max(sizes) - min(s for s in sizes[:-1] or sizes) <= 2 * 256 or V < 256 * R
    # more ranks than vocab tiles: the surplus ranks own no rows (they contribute the merge's neutral element)
    st = sq.shard_vocab(600, 5)
    assert st == [0, 0, 256, 256, 512, 600] and sum(b > a for a, b in zip(st, st[1:])) == 3
    # the packed state's size does not depend on the shard's row count: uneven and empty shards exchange equal blocks
    assert sq.shard_state_bytes(100, 20) == (6 + 40) * 100 * 4


def _vp_worker(rank, world, port, words, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    state = torch.full((words,), float(rank + 1)) + torch.arange(words) * 1e-3      # this rank's packed state
    ret[rank] = sharding.gather_shard_states(state, world).clone()                  # the ONE collective of the path
    dist.barrier()
    dist.destroy_process_group()


def test_vocab_parallel_state_exchange_layout():
    """The merge kernel reads shard r's state at word offset r * words: the gathered tensor must be rank-major."""
    import paper_2604_07725_b200 as sq
    words = sq.shard_state_bytes(7, 5) // 4
    assert words == (6 + 16) * 7
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_vp_worker, args=(2, _free_port(), words, ret), nprocs=2, join=True)
        got = dict(ret)
    for r in range(2):
        g = got[r]
        assert g.shape == (2, words) and g.is_contiguous()
        assert torch.allclose(g[0], torch.full((words,), 1.0) + torch.arange(words) * 1e-3)
        assert torch.allclose(g[1], torch.full((words,), 2.0) + torch.arange(words) * 1e-3)
