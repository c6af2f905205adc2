"""CPU-only checks of the boundary: the C-ABI library builds/loads, exports every symbol that
include/sq_score.h declares, its host-side planning logic is sane, and it fails loudly (never
falls back) when there is no GPU."""
import ctypes
import os
import re

import pytest
import torch

import paper_2604_07725_b200 as sq
from paper_2604_07725_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "sq_score.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sq_score_[a-z_]+)\s*\(", text)))


def test_header_declares_the_named_calls():
    names = declared_functions()
    for required in ("sq_score_create", "sq_score_run", "sq_score_destroy"):   # BASELINE.json north_star
        assert required in names
    assert len(names) >= 10


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    for name in declared_functions():
        assert hasattr(L, name), "libsq_score.so does not export %s" % name
    assert sq.version() >= 100


def test_error_strings():
    L = sq.lib()
    assert L.sq_score_error_string(0) == b"SQ_OK"
    assert L.sq_score_error_string(-1) == b"SQ_ERR_INVALID_ARG"
    assert L.sq_score_error_string(-3) == b"SQ_ERR_CUDA"


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_create_fails_loudly_without_gpu():
    with pytest.raises(sq.SqScoreError) as ei:
        sq.SqScore(64, 1024, 256, 4)
    assert ei.value.code in (sq.ERR_CUDA, sq.ERR_UNSUPPORTED)
    assert "no CPU fallback" in str(ei.value) or "sm_" in str(ei.value)


def test_create_rejects_bad_config_before_touching_cuda():
    L = sq.lib()
    h = ctypes.c_void_p()
    bad = [dict(d=0), dict(vocab=0), dict(max_tokens=0), dict(max_seqs=0), dict(max_k=0), dict(max_k=33), dict(cta_group=3), dict(flags=2)]
    for kw in bad:
        base = dict(device=0, d=64, vocab=1024, max_tokens=256, max_seqs=4, max_k=5, cta_group=0, num_chunks=0, group_m=0, flags=0)
        base.update(kw)
        cfg = binding.sq_score_config(**base)
        assert L.sq_score_create(ctypes.byref(cfg), ctypes.byref(h)) == sq.ERR_INVALID_ARG, kw
        assert h.value is None
    cfg = binding.sq_score_config(device=0, d=60, vocab=1024, max_tokens=256, max_seqs=4, max_k=5)
    assert L.sq_score_create(ctypes.byref(cfg), ctypes.byref(h)) == sq.ERR_UNSUPPORTED      # d % 8 != 0
    assert b"multiple of 8" in L.sq_score_last_error(None)
    assert L.sq_score_create(None, ctypes.byref(h)) == sq.ERR_INVALID_ARG
    assert L.sq_score_destroy(None) == 0


# ------------------------------------------------------------------------------------------ planning
CONFIG_SHAPES = {"tiny": (64, 1024, 256, 5), "qwen3_4b": (2560, 151936, 20480, 20), "qwen3_8b": (4096, 151936, 81920, 20),
                 "gpt_oss": (2880, 201088, 73728, 20), "qwen3_32b": (5120, 151936, 557056, 20)}


@pytest.mark.parametrize("name", list(CONFIG_SHAPES))
@pytest.mark.parametrize("cg", [1, 2])
def test_plan_covers_every_tile_exactly_once(name, cg):
    d, V, T, k = CONFIG_SHAPES[name]
    p = sq.plan(d, V, T, k, num_sms=148, cta_group=cg)
    assert p["cta_group"] == cg and p["rows_per_tile"] == 128 * cg
    assert p["m_tiles"] == -(-T // (128 * cg))
    assert p["num_vtiles"] == -(-V // 256) and p["num_k_blocks"] == -(-d // 64)
    assert 1 <= p["num_chunks"] <= 160
    # chunks tile the vocabulary: no empty chunk, full coverage
    assert p["tiles_per_chunk"] * p["num_chunks"] >= p["num_vtiles"]
    assert p["tiles_per_chunk"] * (p["num_chunks"] - 1) < p["num_vtiles"]
    assert p["num_units"] == p["m_tiles"] * p["num_chunks"]
    assert p["num_clusters"] == 148 // cg
    assert p["topk_cap"] >= k
    # replay the kernel's gang-unit decode (class-A gangs + the smaller gang B): every
    # (m_tile, chunk) pair is visited exactly once
    G, C, M = p["group_m"], p["num_chunks"], p["m_tiles"]
    assert 1 <= G <= max(1, min(M, p["num_clusters"]))
    assert p["num_gangs"] == p["num_clusters"] // G and p["num_gangs"] >= 1
    assert p["gang_b_size"] == p["num_clusters"] - p["num_gangs"] * G
    assert 0 <= p["m_split"] <= M
    assert p["num_gang_units"] == -(-p["m_split"] // G) * C
    seen = set()
    for gang in range(p["num_gangs"]):
        for gu in range(gang, p["num_gang_units"], p["num_gangs"]):
            g, c = divmod(gu, C)
            for member in range(G):
                m = g * G + member
                if m < p["m_split"]:
                    assert (m, c) not in seen
                    seen.add((m, c))
    if p["m_split"] < M:
        GB = p["gang_b_size"]
        assert GB >= 1 and p["num_gang_units_b"] == -(-(M - p["m_split"]) // GB) * C
        for gu in range(p["num_gang_units_b"]):
            g, c = divmod(gu, C)
            for member in range(GB):
                m = p["m_split"] + g * GB + member
                if m < M:
                    assert (m, c) not in seen
                    seen.add((m, c))
    else:
        assert p["num_gang_units_b"] == 0
    assert len(seen) == p["num_units"]


def test_plan_wave_efficiency_on_target_config():
    d, V, T, k = CONFIG_SHAPES["qwen3_8b"]
    p = sq.plan(d, V, T, k, num_sms=148)
    rounds = max(-(-p["num_gang_units"] // p["num_gangs"]), p["num_gang_units_b"])
    ideal = p["m_tiles"] * p["num_vtiles"] / p["num_clusters"]
    assert ideal / (rounds * p["tiles_per_chunk"]) > 0.95    # < 5 % lost to gang/wave quantisation


def test_plan_decode_shaped_defaults():
    p = sq.plan(4096, 151936, 64, 20, num_sms=148)
    assert p["cta_group"] == 1 and p["group_m"] == 1 and p["num_gangs"] == 148 and p["num_chunks"] > 100
    p = sq.plan(4096, 151936, 256, 20, num_sms=148)
    assert p["cta_group"] == 2 and p["num_gangs"] == 74 and 60 <= p["num_chunks"] <= 74


def test_plan_forced_chunks_and_edge_sizes():
    assert sq.plan(64, 1024, 256, 5, num_chunks=2)["num_chunks"] == 2
    assert sq.plan(64, 1024, 256, 5, num_chunks=99)["num_chunks"] == 4        # clamped to the number of vocab tiles
    p = sq.plan(64, 1024, 0, 5)
    assert p["m_tiles"] == 0 and p["num_units"] == 0
    assert sq.plan(64, 100, 1, 1)["num_vtiles"] == 1
    with pytest.raises(sq.SqScoreError):
        sq.plan(64, 1024, 256, 0)
    with pytest.raises(sq.SqScoreError):
        sq.plan(64, 1024, 256, 33)
    assert sq.plan(64, 1024, 256, 8)["topk_cap"] == 8
    assert sq.plan(64, 1024, 256, 9)["topk_cap"] == 20
    assert sq.plan(64, 1024, 256, 21)["topk_cap"] == 32


def test_shard_sequences_balances_and_partitions():
    lens = [5000, 100, 4000, 3000, 2500, 2500, 700, 10]
    for ws in (1, 2, 3, 8):
        parts = sq.shard_sequences(lens, ws)
        flat = sorted(i for p in parts for i in p)
        assert flat == list(range(len(lens)))
        loads = [sum(lens[i] for i in p) for p in parts]
        if ws == 2:
            assert max(loads) - min(loads) <= max(lens)
    assert sq.shard_sequences([], 2) == [[], []]
