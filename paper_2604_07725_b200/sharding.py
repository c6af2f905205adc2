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


def gather_sequence_scores(local: dict, seq_ids: Sequence[int], num_seqs: int, world_size: int, group=None) -> dict:
    """all_gather of the per-sequence scalars into global sequence order.  `local[key]` is a [B_local]
    float tensor on the collective's device."""
    import torch.distributed as dist
    dev = local[SEQ_KEYS[0]].device if len(seq_ids) else torch.device("cpu")
    cap = num_seqs   # a rank can hold at most all sequences
    buf = torch.full((cap, 1 + len(SEQ_KEYS)), float("nan"), dtype=torch.float32, device=dev)
    n = len(seq_ids)
    if n:
        buf[:n, 0] = torch.tensor(list(seq_ids), dtype=torch.float32, device=dev)
        for j, key in enumerate(SEQ_KEYS):
            buf[:n, 1 + j] = local[key].to(torch.float32)
    buf[n:, 0] = -1.0
    gathered = [torch.empty_like(buf) for _ in range(world_size)]
    dist.all_gather(gathered, buf, group=group)
    out = {key: torch.full((num_seqs,), float("nan"), dtype=torch.float32) for key in SEQ_KEYS}
    for g in gathered:
        g = g.cpu()
        for r in range(g.shape[0]):
            b = int(g[r, 0])
            if b >= 0:
                for j, key in enumerate(SEQ_KEYS):
                    out[key][b] = g[r, 1 + j]
    return out


def score_vocab_parallel(eng, H, W_shard, vocab_starts: Sequence[int], rank: int, targets, cu_seqlens, k: int, window: int,
                         group=None, stream=None) -> dict:
    """Vocab-parallel scoring on one rank: this rank's shard of the LM head -> packed partial
    state, ONE all_gather of the states (NCCL over NVLink on GPUs), then the associative merge + kernel 2 on every
    rank.  `eng` was created with vocab = the largest shard; every rank passes the same H, targets and cu_seqlens."""
    import torch.distributed as dist
    world = len(vocab_starts) - 1
    if vocab_starts[rank + 1] > vocab_starts[rank]:
        state = eng.run_shard(H, W_shard, vocab_starts[rank], targets, k, stream=stream)
    else:                                                  # more ranks than vocab tiles: this rank owns no rows
        from .binding import neutral_shard_state
        state = neutral_shard_state(H.shape[0], k, H.device)
    states = gather_shard_states(state, world, group=group, stream=stream)
    return eng.merge_shards(states, vocab_starts, targets, cu_seqlens, k, window, stream=stream)


def gather_shard_states(state: torch.Tensor, world_size: int, group=None, stream=None) -> torch.Tensor:
    """The one collective of the vocab-parallel path: all_gather of the packed states, rank-major -- shard r's state
    starts r * words into the result, which is what sq_score_merge_shards reads."""
    import torch.distributed as dist
    flat = torch.empty(world_size * state.numel(), dtype=state.dtype, device=state.device)
    if stream is not None:
        stream.synchronize()   # the collective runs on its own stream
    dist.all_gather_into_tensor(flat, state, group=group)
    return flat.view(world_size, state.numel())
