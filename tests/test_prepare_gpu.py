"""GPU parity of the step before the path: sq_score_prepare (gather of the predicting
positions + final RMSNorm) and sq_score_run_x, against the fp64 oracle.

H is a quantised code (bf16), decided by floating point.  The kernel computes in fp32 (sum of squares over
d <= 8192 terms, one division, one square root, two multiplies), so its unrounded value is within
32 * 2^-24 relative of the exact one; the GPU's bf16 must therefore lie within half a bf16 ulp of the
oracle's fp64 value widened by that much -- i.e. it is a correct rounding of a value that close -- and it
must EQUAL the oracle's own rounding except where the exact value sits that close to a rounding boundary."""
import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O
from test_parity_gpu import check_seqs, check_tokens

pytestmark = pytest.mark.gpu
FP32_SLACK = 32 * 2.0 ** -24


def _sq():
    import paper_2604_07725_b200 as sq
    return sq


def check_prepared(H_gpu, h64):
    got = H_gpu.double().cpu().numpy()
    err = np.abs(got - h64)
    lim = O.bf16_half_ulp(h64) + FP32_SLACK * np.abs(h64)
    assert (err <= lim).all(), "worst excess %g at %s" % ((err - lim).max(), np.unravel_index((err - lim).argmax(), err.shape))
    ref = O.round_to_bf16(h64).double().numpy()
    diff = got != ref
    if diff.any():   # only at values that sit on a rounding boundary to within the fp32 slack
        near = np.abs(np.abs(h64 - ref) - O.bf16_half_ulp(h64)) <= 2 * FP32_SLACK * np.abs(h64) + 1e-300
        assert near[diff].all()
    assert diff.mean() < 1e-3


@pytest.mark.parametrize("d,N,T", [(64, 50, 37), (200, 300, 300), (4096, 700, 513), (5120, 64, 200), (8, 5, 9), (8192, 40, 33)])
def test_prepare_matches_oracle(d, N, T):
    sq = _sq()
    gen = torch.Generator().manual_seed(d + N)
    scale = torch.exp(torch.rand(N, 1, generator=gen) * 3 - 1)
    X = (torch.randn(N, d, generator=gen) * scale).to(torch.bfloat16)
    gain = (1 + 0.1 * torch.randn(d, generator=gen)).to(torch.bfloat16)
    pos = torch.randint(0, N, (T,), generator=gen, dtype=torch.int32)
    pos[0] = 0; pos[-1] = N - 1
    eng = sq.SqScore(d, 1000, max_tokens=max(T, N), max_seqs=1)
    dev = torch.device("cuda:0")
    H = eng.prepare(X.to(dev), pos.to(dev), gain.to(dev), 1e-6)
    torch.cuda.synchronize()
    check_prepared(H, O.prepare_hidden(X, pos.numpy(), gain, 1e-6))
    # identity positions, and in place
    Xd = X.to(dev).clone()
    H2 = eng.prepare(Xd, None, gain.to(dev), 1e-5, out=Xd)
    torch.cuda.synchronize()
    assert H2.data_ptr() == Xd.data_ptr()
    check_prepared(H2, O.prepare_hidden(X, np.arange(N), gain, 1e-5))
    eng.close()


def test_prepare_special_rows():
    sq = _sq()
    d = 256
    X = torch.zeros(4, d, dtype=torch.bfloat16)
    X[1] = 2.5; X[2] = -2.5; X[3, 7] = 3.0
    gain = torch.ones(d, dtype=torch.bfloat16)
    eng = sq.SqScore(d, 1000, max_tokens=8, max_seqs=1)
    dev = torch.device("cuda:0")
    H = eng.prepare(X.to(dev), torch.tensor([0, 1, 2, 3, 1], dtype=torch.int32, device=dev), gain.to(dev), 1e-6).cpu().float()
    assert (H[0] == 0).all()                                   # zero row: 0 / sqrt(eps) = 0
    assert (H[1] == 1).all() and (H[2] == -1).all()            # constant rows normalise to +-1
    assert H[3, 7] == 16.0 and H[3].abs().sum() == 16.0        # one-hot 3 -> 3 / sqrt(9/256) = 16
    assert torch.equal(H[4], H[1])                             # a row gathered twice is bit-identical
    Xd = X.to(dev)
    with pytest.raises(sq.SqScoreError):       # gathering in place would read rows already overwritten
        eng.prepare(Xd, torch.tensor([0], dtype=torch.int32, device=dev), gain.to(dev), 1e-6, out=Xd)
    eng.close()


def test_run_x_end_to_end_against_oracle():
    sq = _sq()
    wl = workloads.custom(d=200, V=1003, B=3, len_lo=20, len_hi=150, k=5, window=16, seed=21)
    inp = workloads.prepare_inputs(wl, query_lo=1, query_hi=40)
    pos, cu = O.trajectory_positions(inp["query_lens"], inp["traj_lens"])
    pos_b, cu_b = sq.trajectory_positions(inp["query_lens"].tolist(), inp["traj_lens"].tolist())
    assert pos_b == pos.tolist() and cu_b == cu.tolist()
    dev = torch.device("cuda:0")
    eng = sq.SqScore(wl.d, wl.V, max_tokens=inp["T"], max_seqs=inp["B"], max_k=wl.k, staging=True)
    Xd, Wd, gd = inp["X"].to(dev), inp["W"].to(dev), inp["gain"].to(dev)
    # the position list comes from the device kernel (no host round trip) and must equal the oracle's
    pd, cd, status = eng.positions(inp["query_lens"].to(torch.int32).to(dev), inp["traj_lens"].to(torch.int32).to(dev), inp["T"],
                                   with_status=True)
    torch.cuda.synchronize()
    assert pd.cpu().tolist() == pos.tolist() and cd.cpu().tolist() == cu.tolist() and int(status) == 0
    td = inp["targets"].to(dev)
    out = eng.run_x(Xd, pd, gd, inp["eps"], Wd, td, cd, wl.k, wl.window)
    torch.cuda.synchronize()
    # (1) run_x == prepare + run, bit for bit
    Hd = eng.prepare(Xd, pd, gd, inp["eps"])
    out2 = eng.run(Hd, Wd, td, cd, wl.k, wl.window)
    torch.cuda.synchronize()
    for n in out:
        assert torch.equal(out[n], out2[n]) or (torch.isnan(out[n]) == torch.isnan(out2[n])).all(), n
    # (2) the prepared H is the oracle's up to the rounding criterion
    h64 = O.prepare_hidden(inp["X"], pos, inp["gain"], inp["eps"])
    check_prepared(Hd, h64)
    # (3) the scores match the oracle run end to end from X (H rounded by the oracle itself)
    ref = O.score(O.round_to_bf16(h64), inp["W"], inp["targets"], cu, wl.k, wl.window)
    o = {n: v.cpu().numpy() for n, v in out.items()}
    check_tokens(o, ref, wl.k)
    check_seqs(o, ref)
    eng.close()


@pytest.mark.parametrize("B,qr,nr", [(1, (1, 1), (1, 1)), (7, (1, 40), (0, 300)), (1500, (1, 9), (0, 50)), (4096, (1, 3), (0, 7)), (3, (5, 5), (0, 0))])
def test_positions_kernel_matches_oracle(B, qr, nr):
    """sq_score_positions (device) against the oracle's trajectory_positions: many candidates (the scan spans several
    candidates per thread), empty trajectories, an all-empty batch; and the status word for bad inputs."""
    sq = _sq()
    rng = np.random.default_rng(B)
    q = rng.integers(qr[0], qr[1] + 1, size=B); n = rng.integers(nr[0], nr[1] + 1, size=B)
    pos, cu = O.trajectory_positions(q, n)
    dev = torch.device("cuda:0")
    eng = sq.SqScore(64, 1000, max_tokens=max(1, len(pos)), max_seqs=B)
    pd, cd, st = eng.positions(torch.tensor(q, dtype=torch.int32, device=dev), torch.tensor(n, dtype=torch.int32, device=dev), len(pos),
                               with_status=True)
    torch.cuda.synchronize()
    assert pd.cpu().tolist() == pos.tolist() and cd.cpu().tolist() == cu.tolist() and int(st) == 0
    if B >= 7 and n.sum() > 0:
        q2 = q.copy(); b = int(np.argmax(n > 0)); q2[b] = 0                  # a trajectory with no query token before it
        _, _, st2 = eng.positions(torch.tensor(q2, dtype=torch.int32, device=dev), torch.tensor(n, dtype=torch.int32, device=dev), len(pos),
                                  with_status=True)
        _, _, st3 = eng.positions(torch.tensor(q, dtype=torch.int32, device=dev), torch.tensor(n, dtype=torch.int32, device=dev), len(pos) - 1,
                                  with_status=True)                           # lengths that do not sum to num_tokens
        torch.cuda.synchronize()
        assert int(st2) == 1 and int(st3) == 1
    eng.close()


def test_prepare_full_size_rows_sampled():
    """qwen3_8b-shaped d at a size that spans many CTAs and the grid-stride loop; the oracle checks a row sample."""
    sq = _sq()
    d, N = 4096, 40000
    gen = torch.Generator().manual_seed(77)
    X = torch.empty(N, d, dtype=torch.bfloat16)
    for r0 in range(0, N, 8192):
        r1 = min(N, r0 + 8192)
        X[r0:r1] = (torch.randn(r1 - r0, d, generator=gen) * torch.exp(torch.rand(r1 - r0, 1, generator=gen) * 3 - 1)).to(torch.bfloat16)
    gain = (1 + 0.1 * torch.randn(d, generator=gen)).to(torch.bfloat16)
    T = 30001
    pos = torch.randint(0, N, (T,), generator=gen, dtype=torch.int32)
    dev = torch.device("cuda:0")
    eng = sq.SqScore(d, 1000, max_tokens=T, max_seqs=1)
    H = eng.prepare(X.to(dev), pos.to(dev), gain.to(dev), 1e-6)
    torch.cuda.synchronize()
    rows = np.unique(np.concatenate([[0, 1, 7, 8, T - 1, T - 2], np.random.default_rng(1).integers(0, T, 200)]))
    check_prepared(H[torch.as_tensor(rows, device=dev)], O.prepare_hidden(X, pos.numpy()[rows], gain, 1e-6))
    eng.close()
