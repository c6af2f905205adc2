"""sq_score -- B200-native fused LM-head scoring (SQUEEZE EVOLVE confidence path, Eq. 3 / Eq. 4).

Thin ctypes binding over the C ABI in include/sq_score.h.  Argument marshalling only: every step
of the path runs in the CUDA kernels of csrc/.  There is no CPU fallback.
"""
from .binding import (SqScore, SqScoreError, plan, lib, version, shard_sequences, trajectory_positions, shard_vocab, shard_state_bytes,  # noqa: F401
                      reduce_static, STATIC_MAX_TOKENS, STATIC_MAX_SEQS, SQ_MAX_K, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_NOMEM, MX_OPERAND_H, MX_OPERAND_W)
