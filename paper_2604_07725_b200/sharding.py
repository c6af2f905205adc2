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
    if rows > 0:
        state = eng.run_shard(H, W_shard, vocab_starts[rank], targets, k, stream=stream)
    else:                                                  # more ranks than vocab tiles: this rank owns no rows
        state = eng.neutral_shard_state(H.shape[0], k, device=H.device, stream=stream)
    states = gather_shard_states(state, world, group=group, stream=stream)
    return eng.merge_shards(states, vocab_starts, targets, cu_seqlens, k, window, stream=stream)


def gather_shard_states(state: torch.Tensor, world_size: int, group=None, stream=None) -> torch.Tensor:
    """The one collective of the vocab-parallel path: all_gather of the packed states, rank-major -- shard r's state
    starts r * words into the result, which is what sq_score_merge_shards reads.  On CUDA the collective is issued
    with `stream` current, so it is ordered after the shard kernels and before the merge on that stream by stream
    order alone: no host synchronisation."""
    import torch.distributed as dist
    flat = torch.empty(world_size * state.numel(), dtype=state.dtype, device=state.device)
    if state.is_cuda:
        with torch.cuda.stream(stream if stream is not None else torch.cuda.current_stream(state.device)):
            dist.all_gather_into_tensor(flat, state, group=group)
    else:
        dist.all_gather_into_tensor(flat, state, group=group)
    return flat.view(world_size, state.numel())
