"""Multi-GPU plumbing: whole sequences are dealt to ranks, W is replicated,
each rank runs sq_score_run on its own packed sub-batch -- no collective on the data path.  The only
exchange is one all_gather of the 4 scalars per sequence at the end (NCCL on GPUs, gloo in tests)."""
from __future__ import annotations

from typing import List, Sequence, Tuple

import torch

from .binding import shard_sequences

SEQ_KEYS = ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")


def local_batch(cu_seqlens: torch.Tensor, rank: int, world_size: int) -> Tuple[List[int], torch.Tensor, torch.Tensor]:
    """Returns (global ids of this rank's sequences, local cu_seqlens int32, global row index of
    every local token in packed order)."""
    cu = cu_seqlens.to(torch.int64).cpu()
    lengths = (cu[1:] - cu[:-1]).tolist()
    mine = shard_sequences(lengths, world_size)[rank]
    local_cu = torch.zeros(len(mine) + 1, dtype=torch.int64)
    rows = []
    for i, b in enumerate(mine):
        local_cu[i + 1] = local_cu[i] + lengths[b]
        rows.append(torch.arange(int(cu[b]), int(cu[b + 1]), dtype=torch.int64))
    row_index = torch.cat(rows) if rows else torch.zeros(0, dtype=torch.int64)
    return mine, local_cu.to(torch.int32), row_index


def gather_sequence_scores(local: dict, seq_ids: Sequence[int], num_seqs: int, world_size: int, group=None,
                           device=None) -> dict:
    """The one exchange of the data-parallel path: all_gather of the per-sequence scalars into global sequence
    order, on the collective's device (`device`: cuda under NCCL, cpu under gloo; default = where `local` lives).
    Every rank sends one packed [num_seqs, 1 + 4] block (sequence id, 4 scalars; unused rows carry id -1) in ONE
    all_gather_into_tensor, and the result is scattered by id with tensor ops -- no host round trip, no per-row
    loop.  `local[key]` is a [B_local] float tensor."""
    import torch.distributed as dist
    if device is None:
        device = local[SEQ_KEYS[0]].device
    device = torch.device(device)
    n = len(seq_ids)
    buf = torch.full((num_seqs, 1 + len(SEQ_KEYS)), float("nan"), dtype=torch.float32, device=device)
    buf[:, 0] = -1.0
    if n:
        buf[:n, 0] = torch.as_tensor(list(seq_ids), dtype=torch.float32, device=device)
        buf[:n, 1:] = torch.stack([local[key].to(device=device, dtype=torch.float32) for key in SEQ_KEYS], dim=1)
    flat = torch.empty((world_size * num_seqs, 1 + len(SEQ_KEYS)), dtype=torch.float32, device=device)
    dist.all_gather_into_tensor(flat, buf, group=group)
    ids = flat[:, 0].to(torch.int64)
    keep = ids >= 0
    table = torch.full((num_seqs, len(SEQ_KEYS)), float("nan"), dtype=torch.float32, device=device)
    table[ids[keep]] = flat[keep, 1:]
    return {key: table[:, j] for j, key in enumerate(SEQ_KEYS)}


def score_vocab_parallel(eng, H, W_shard, vocab_starts: Sequence[int], rank: int, targets, cu_seqlens, k: int, window: int,
                         group=None, stream=None) -> dict:
    """Vocab-parallel scoring on one rank: this rank's shard of the LM head -> packed partial
    state, ONE all_gather of the states (NCCL over NVLink on GPUs), then the associative merge + kernel 2 on every
    rank.  `eng` was created with vocab >= the LARGEST shard (sq_score_run_shard takes this rank's own row count from
    W_shard); every rank passes the same H, targets and cu_seqlens."""
    world = len(vocab_starts) - 1
    rows = int(vocab_starts[rank + 1]) - int(vocab_starts[rank])
    if rows != W_shard.shape[0]:
        raise ValueError("W_shard has %d rows, vocab_starts gives this rank %d" % (W_shard.shape[0], rows))

    def step():
        if rows > 0:
            state = eng.run_shard(H, W_shard, vocab_starts[rank], targets, k, stream=stream)
        else:                                              # more ranks than vocab tiles: this rank owns no rows
            state = eng.neutral_shard_state(H.shape[0], k, device=H.device, stream=stream)
        states = gather_shard_states(state, world, group=group, stream=stream)
        return eng.merge_shards(states, vocab_starts, targets, cu_seqlens, k, window, stream=stream)

    # The packed state, the gathered states and the outputs are allocated here and used by kernels on `stream`: with
    # `stream` current the caching allocator ties those blocks to it, so a block freed when this function returns is not
    # handed to another stream's tensor while kernels on `stream` still read or write it.
    if stream is not None and H.is_cuda:
        with torch.cuda.stream(stream):
            return step()
    return step()


class PeerStates:
    """The vocab-parallel exchange WITHOUT an all-gather: every rank keeps its packed state in
    a buffer of its own, the ranks open one another's buffers once (CUDA IPC; over NVLink a peer's buffer is ordinary
    device memory to a kernel), and sq_score_merge_shards_peer reads all R states in place -- the transfer is the merge
    kernel's own loads.  Per step the ranks only have to agree on WHEN: `ready()` after the shard kernels (nobody reads a
    state before it is written) and `release()` after the merge (nobody overwrites a state a peer may still be reading).
    Under NCCL both are a 4-byte all-reduce enqueued on the compute stream -- ordered by the stream, no host
    synchronisation; under gloo (CPU-side groups, the one-GPU test) the stream is synchronised and the ranks meet at a
    host barrier."""

    def __init__(self, state: torch.Tensor, rank: int, world_size: int, group=None):
        import torch.distributed as dist
        from torch.multiprocessing.reductions import reduce_tensor
        self.rank, self.world, self.group = rank, world_size, group
        self.state = state                                   # this rank's buffer: sq_score_run_shard writes into it every step
        self._nccl = dist.get_backend(group) == "nccl"
        self._flag = torch.zeros(1, dtype=torch.int32, device=state.device)
        handles = [None] * world_size
        dist.all_gather_object(handles, reduce_tensor(state), group=group)
        self.views = []
        for r, (rebuild, args) in enumerate(handles):
            if r == rank:
                self.views.append(state)
                continue
            v = rebuild(*args)                               # maps the peer's allocation into this process
            if v.device != state.device:                     # another GPU: one element through torch's P2P path enables peer access
                torch.empty(1, dtype=v.dtype, device=state.device).copy_(v[:1])
            self.views.append(v)

    def _meet(self, stream):
        import torch.distributed as dist
        if self._nccl:
            with torch.cuda.stream(stream if stream is not None else torch.cuda.current_stream(self.state.device)):
                dist.all_reduce(self._flag, group=self.group)
        else:
            (stream if stream is not None else torch.cuda.current_stream(self.state.device)).synchronize()
            dist.barrier(group=self.group)

    def close(self):
        """Drops the mappings of the peers' buffers (call on every rank before the buffers are freed)."""
        self.views = []

    def ready(self, stream=None):
        self._meet(stream)

    def release(self, stream=None):
        self._meet(stream)


def score_vocab_parallel_peer(eng, peers: PeerStates, H, W_shard, vocab_starts: Sequence[int], targets, cu_seqlens, k: int,
                              window: int, stream=None) -> dict:
    """score_vocab_parallel with the peers' states read in place (PeerStates) instead of gathered: shard kernels ->
    ready() -> merge over peer memory + kernel 2 -> release()."""
    rank = peers.rank
    rows = int(vocab_starts[rank + 1]) - int(vocab_starts[rank])
    if rows != W_shard.shape[0]:
        raise ValueError("W_shard has %d rows, vocab_starts gives this rank %d" % (W_shard.shape[0], rows))
    if rows > 0:
        eng.run_shard(H, W_shard, vocab_starts[rank], targets, k, out=peers.state, stream=stream)
    else:
        eng.neutral_shard_state(H.shape[0], k, device=H.device, stream=stream, out=peers.state)
    peers.ready(stream)
    out = eng.merge_shards_peer(peers.views, vocab_starts, targets, cu_seqlens, k, window, stream=stream)
    peers.release(stream)
    return out


def gather_shard_states(state: torch.Tensor, world_size: int, group=None, stream=None) -> torch.Tensor:
    """The one collective of the vocab-parallel path: all_gather of the packed states, rank-major -- shard r's state
    starts r * words into the result, which is what sq_score_merge_shards reads.  On CUDA the collective is issued
    with `stream` current, so it is ordered after the shard kernels and before the merge on that stream by stream
    order alone: no host synchronisation."""
    import torch.distributed as dist
    if state.is_cuda:
        s = stream if stream is not None else torch.cuda.current_stream(state.device)
        with torch.cuda.stream(s):
            # allocated with `s` current (see score_vocab_parallel); `state` may come from another stream's pool
            flat = torch.empty(world_size * state.numel(), dtype=state.dtype, device=state.device)
            dist.all_gather_into_tensor(flat, state, group=group)
        state.record_stream(s)
    else:
        flat = torch.empty(world_size * state.numel(), dtype=state.dtype, device=state.device)
        dist.all_gather_into_tensor(flat, state, group=group)
    return flat.view(world_size, state.numel())
