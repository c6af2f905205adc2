"""Pins for the oracle's 8(f)-2 functions (gather of the predicting positions + final RMSNorm):
hand values, invariants, a library routine on the special case it covers, and brute force.
-m "not gpu"."""
import math

import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O


def bf(x):
    return torch.tensor(x, dtype=torch.float32).to(torch.bfloat16)


def test_positions_hand_case():
    # candidate 0: 3 query + 2 trajectory tokens -> packed rows 0..4; candidate 1: 1 query + 3 trajectory -> rows 5..8
    pos, cu = O.trajectory_positions([3, 1], [2, 3])
    assert pos.tolist() == [2, 3, 5, 6, 7]      # the state BEFORE each trajectory token ("t_<i, Q")
    assert cu.tolist() == [0, 2, 5]             # only trajectory tokens are scored


def test_positions_brute_force_and_edges():
    rng = np.random.default_rng(5)
    for _ in range(20):
        B = int(rng.integers(1, 6))
        q = rng.integers(1, 9, B); L = rng.integers(0, 9, B)
        pos, cu = O.trajectory_positions(q, L)
        # brute force: label every packed position, then pick "previous position of every trajectory token"
        labels = []
        for b in range(B):
            labels += [("q", b)] * int(q[b]) + [("t", b)] * int(L[b])
        want = [i - 1 for i, (kind, _) in enumerate(labels) if kind == "t"]
        assert pos.tolist() == want
        assert np.diff(cu).tolist() == L.tolist()
        for t, p in enumerate(pos):            # the predicting state belongs to the same candidate
            b = int(np.searchsorted(cu, t, side="right") - 1)
            assert labels[p][1] == b
    with pytest.raises(ValueError):
        O.trajectory_positions([0], [4])
    pos, cu = O.trajectory_positions([0, 2], [0, 1])   # an empty candidate without a query is fine
    assert pos.tolist() == [1] and cu.tolist() == [0, 0, 1]


def test_rmsnorm_hand_values():
    X = bf([[3.0, 4.0], [1.0, 1.0]])
    g = bf([1.0, 2.0])
    h = O.prepare_hidden(X, [0, 1, 0], g, 0.0)
    r = math.sqrt(12.5)
    assert np.allclose(h[0], [3.0 / r, 8.0 / r], rtol=0, atol=1e-15)
    assert np.allclose(h[1], [1.0, 2.0], rtol=0, atol=1e-15)
    assert np.array_equal(h[2], h[0])                      # gathering a row twice
    h = O.prepare_hidden(X, [0], g, 12.5)                  # eps inside the square root, added to the MEAN square
    assert np.allclose(h[0], [3.0 / 5.0, 8.0 / 5.0], rtol=0, atol=1e-15)


def test_rmsnorm_invariants():
    gen = torch.Generator().manual_seed(3)
    X = (torch.randn(9, 40, generator=gen) * 3).to(torch.bfloat16)
    one = torch.ones(40, dtype=torch.bfloat16)
    h = O.prepare_hidden(X, np.arange(9), one, 0.0)
    assert np.allclose((h * h).mean(axis=1), 1.0, atol=1e-14)             # unit gain, eps = 0: unit mean square
    X4 = (X.float() * 4).to(torch.bfloat16)                                  # exact power-of-two scaling
    assert np.allclose(O.prepare_hidden(X4, np.arange(9), one, 0.0), h, atol=1e-14)   # scale invariance
    g = (1 + 0.1 * torch.randn(40, generator=gen)).to(torch.bfloat16)
    hg = O.prepare_hidden(X, np.arange(9), g, 0.0)
    assert np.allclose(hg, h * g.double().numpy()[None, :], atol=1e-14)    # the gain is a per-column factor
    perm = np.array([4, 0, 8, 8, 2])
    assert np.array_equal(O.prepare_hidden(X, perm, g, 1e-6), O.prepare_hidden(X, np.arange(9), g, 1e-6)[perm])
    c = bf([[2.5] * 16])
    assert np.allclose(O.prepare_hidden(c, [0], torch.ones(16, dtype=torch.bfloat16), 0.0), 1.0, atol=1e-15)
    c = bf([[-2.5] * 16])
    assert np.allclose(O.prepare_hidden(c, [0], torch.ones(16, dtype=torch.bfloat16), 0.0), -1.0, atol=1e-15)


def test_rmsnorm_matches_library_routine():
    gen = torch.Generator().manual_seed(4)
    X = torch.randn(6, 64, generator=gen).to(torch.bfloat16)
    g = (1 + 0.1 * torch.randn(64, generator=gen)).to(torch.bfloat16)
    ref = torch.nn.functional.rms_norm(X.double(), (64,), weight=g.double(), eps=1e-6).numpy()
    assert np.allclose(O.prepare_hidden(X, np.arange(6), g, 1e-6), ref, rtol=1e-14, atol=1e-15)


def test_rmsnorm_brute_force_python():
    gen = torch.Generator().manual_seed(6)
    X = torch.randn(4, 7, generator=gen).to(torch.bfloat16)
    g = torch.randn(7, generator=gen).to(torch.bfloat16)
    pos = [3, 1, 1]
    h = O.prepare_hidden(X, pos, g, 1e-5)
    for t, p in enumerate(pos):
        xs = [float(X[p, j]) for j in range(7)]
        ms = sum(v * v for v in xs) / 7
        for j in range(7):
            assert abs(h[t, j] - xs[j] / math.sqrt(ms + 1e-5) * float(g[j])) < 1e-14


def test_bf16_rounding_helpers():
    v = np.array([1.0, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -9, -3.0, 0.1])
    r = O.round_to_bf16(v).double().numpy()
    assert r[0] == 1.0 and r[1] == 1.0 and r[2] == 1.0 + 2.0 ** -7 and r[3] == -3.0     # ties to even, exact values
    assert np.all(np.abs(r - v) <= O.bf16_half_ulp(v))
    assert O.bf16_half_ulp(np.array([1.0]))[0] == 2.0 ** -8 and O.bf16_half_ulp(np.array([3.9]))[0] == 2.0 ** -7


def test_prepare_inputs_recipe_is_seeded_and_shaped():
    wl = workloads.custom(d=64, V=300, B=3, len_lo=5, len_hi=20, seed=11)
    a = workloads.prepare_inputs(wl, query_lo=2, query_hi=6)
    b = workloads.prepare_inputs(wl, query_lo=2, query_hi=6)
    assert torch.equal(a["X"], b["X"]) and torch.equal(a["gain"], b["gain"])
    assert a["X"].shape == (a["N"], 64) and a["N"] == int(a["traj_lens"].sum() + a["query_lens"].sum())
    pos, cu = O.trajectory_positions(a["query_lens"], a["traj_lens"])
    assert len(pos) == a["T"] and pos.max() < a["N"] - 1 + 1 and pos.min() >= 0
    rms = a["X"].double().pow(2).mean(dim=1).sqrt()
    assert 0.3 < float(rms.min()) and float(rms.max()) < 12.0 and float(rms.max() / rms.min()) > 2.0
