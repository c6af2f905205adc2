"""GPU parity of the routing row against the oracle: GC(g) and theta_q
against the fp64 definitions (rel 1e-6: they are means / interpolations of fp32 inputs), routing
codes bit-exact against the oracle's decision taken in the kernel's precision (fp32), selection
probabilities rel 1e-5.  Also the end of the whole path: sq_score_run's C(tau) fed straight into
sq_score_route on the device."""
import numpy as np
import pytest
import torch

import workloads
from oracle import sq_oracle as O

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _eng(**kw):
    import paper_2604_07725_b200 as sq
    args = dict(d=64, vocab=1024, max_tokens=256, max_seqs=8, max_k=5, reduce_only=True)
    args.update(kw)
    return sq.SqScore(args.pop("d"), args.pop("vocab"), **args)


def make_problems(rng, Q, n_lo, n_hi, m_lo, m_hi, K):
    """Q problems with N_q candidates and M_q groups of K members drawn from the problem's own population."""
    pops = rng.integers(n_lo, n_hi + 1, size=Q)
    pop_off = np.concatenate([[0], np.cumsum(pops)])
    ms = rng.integers(m_lo, m_hi + 1, size=Q)
    grp_off = np.concatenate([[0], np.cumsum(ms)])
    members = np.concatenate([rng.integers(0, pops[q], size=(ms[q], K)) + pop_off[q] for q in range(Q)]) if Q else np.zeros((0, K), int)
    conf = (rng.uniform(3, 12, size=pop_off[-1]) + np.repeat(rng.normal(scale=2, size=Q), pops)).astype(np.float32)
    return conf, members.astype(np.int32), grp_off.astype(np.int32), pop_off.astype(np.int32)


@pytest.mark.parametrize("Q,n,m,K,p,lite_frac", [
    (1, (16, 16), (16, 16), 4, 50.0, 0.0),        # the paper's default: N = 16, K = 4
    (37, (16, 16), (1, 40), 4, 30.0, 0.2),
    (5, (128, 128), (1024, 1024), 4, 50.0, 0.0),  # circle-packing sized population, the sort's capacity
    (64, (4, 4), (1, 3), 2, 70.0, 0.5),
    (9, (8, 32), (5, 300), 1, 0.0, 0.1),
    (9, (8, 32), (5, 300), 7, 100.0, 0.1),
])
def test_route_matches_oracle(Q, n, m, K, p, lite_frac):
    rng = np.random.default_rng(Q * 1000 + K)
    conf, members, grp_off, _ = make_problems(rng, Q, n[0], n[1], m[0], m[1], K)
    G = members.shape[0]
    lite = (rng.uniform(size=G) < lite_frac).astype(np.uint8) if lite_frac > 0 else None
    eng = _eng()
    out = eng.route(torch.tensor(conf, device=DEV), torch.tensor(members, device=DEV), torch.tensor(grp_off, device=DEV), p,
                    lite_mask=None if lite is None else torch.tensor(lite, device=DEV))
    torch.cuda.synchronize()
    ref = O.route(conf, members, grp_off, p, lite)
    np.testing.assert_allclose(out["group_fitness"].cpu().numpy(), ref["group_fitness"], rtol=1e-6)
    th = out["theta"].cpu().numpy()
    assert (np.isnan(th) == np.isnan(ref["theta"])).all()
    np.testing.assert_allclose(th[~np.isnan(th)], ref["theta"][~np.isnan(th)], rtol=1e-6)
    code = out["route"].cpu().numpy()
    assert (code == O.route_decisions_fp32(conf, members, grp_off, p, lite)).all()       # bit-exact in fp32
    far = np.abs(ref["group_fitness"] - np.repeat(ref["theta"], np.diff(grp_off))) > 1e-4
    far &= ~np.isnan(np.repeat(ref["theta"], np.diff(grp_off)))
    assert (code[far] == ref["route"][far]).all()                                         # and equal to fp64 away from ties
    if lite is not None:
        assert (code[lite.astype(bool)] == 0).all()
    eng.close()


def test_route_edge_cases():
    eng = _eng()
    conf = torch.tensor([3.0, 3.0, 3.0, 5.0], device=DEV)
    # problem 0: three identical groups (nothing is strictly above theta -> all Model 2); problem 1: empty;
    # problem 2: one group, lite -> NaN threshold
    members = torch.tensor([[0], [1], [2], [3]], dtype=torch.int32, device=DEV)
    off = torch.tensor([0, 3, 3, 4], dtype=torch.int32, device=DEV)
    lite = torch.tensor([0, 0, 0, 1], dtype=torch.uint8, device=DEV)
    out = eng.route(conf, members, off, 50.0, lite_mask=lite)
    torch.cuda.synchronize()
    assert out["route"].cpu().tolist() == [2, 2, 2, 0]
    th = out["theta"].cpu().numpy()
    assert th[0] == 3.0 and np.isnan(th[1]) and np.isnan(th[2])
    import paper_2604_07725_b200 as sq
    with pytest.raises(sq.SqScoreError):
        eng.route(conf, members, off, 101.0)
    with pytest.raises(sq.SqScoreError) as ei:
        eng.route(conf, members, off, 50.0, max_groups_per_problem=1025)
    assert ei.value.code == sq.ERR_UNSUPPORTED
    eng.close()


@pytest.mark.parametrize("zeta", [0.5, 1.0, 25.0])
def test_select_prob_matches_oracle(zeta):
    rng = np.random.default_rng(5)
    conf, _, _, pop_off = make_problems(rng, 23, 1, 300, 1, 1, 1)
    eng = _eng()
    pr = eng.select_prob(torch.tensor(conf, device=DEV), torch.tensor(pop_off, device=DEV), zeta).cpu().numpy()
    ref = O.selection_probabilities(conf, pop_off, zeta)
    np.testing.assert_allclose(pr, ref, rtol=2e-5, atol=1e-30)
    sums = np.add.reduceat(pr, pop_off[:-1])
    np.testing.assert_allclose(sums, 1.0, rtol=1e-5)
    eng.close()


def test_scores_to_routing_on_device():
    """The whole chain with no host round trip: sq_score_run -> seq_mean_conf = C(tau) -> sq_score_route."""
    import paper_2604_07725_b200 as sq
    wl = workloads.custom(name="pop", d=64, V=1024, B=16, len_lo=20, len_hi=60, k=5, window=8, seed=77, w_std=0.3)
    inp = workloads.make_inputs(wl)                          # one problem, N = 16 candidates
    rng = np.random.default_rng(9)
    members = np.stack([rng.choice(16, size=4, replace=False) for _ in range(16)]).astype(np.int32)   # M = 16 uniform K-subsets
    off = np.array([0, 16], dtype=np.int32)
    eng = sq.SqScore(wl.d, wl.V, max_tokens=inp["T"], max_seqs=16, max_k=5)
    out = eng.run(inp["H"].to(DEV), inp["W"].to(DEV), inp["targets"].to(DEV), inp["cu_seqlens"].to(DEV), 5, 8)
    r = eng.route(out["seq_mean_conf"], torch.tensor(members, device=DEV), torch.tensor(off, device=DEV), 50.0)
    torch.cuda.synchronize()
    tok = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], 5, 8)
    ref = O.route(tok["seq_mean_conf"], members, off, 50.0)
    np.testing.assert_allclose(r["group_fitness"].cpu().numpy(), ref["group_fitness"], rtol=1e-3)
    np.testing.assert_allclose(r["theta"].cpu().numpy(), ref["theta"], rtol=1e-3)
    code = r["route"].cpu().numpy()
    far = np.abs(ref["group_fitness"] - ref["theta"][0]) > 1e-3 * abs(ref["theta"][0])
    assert (code[far] == ref["route"][far]).all()
    assert (code == 1).sum() + (code == 2).sum() == 16 and abs((code == 2).sum() - 8) <= 1
    eng.close()
