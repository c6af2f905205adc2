"""GPU parity of the routing row against the oracle's fp64 definitions.

GC(g) and theta_q: rel 1e-6 (means / interpolations of fp32 inputs).  The routing code is an integer decided
by the floating-point comparison GC(g) > theta_q, which the kernel takes in fp32; it is judged three ways, none
of which mirrors the kernel's operation order:
  (1) it is exactly the comparison of the kernel's OWN reported fp32 GC(g) and theta_q (both already checked
      against fp64);
  (2) it equals the fp64 decision wherever |GC - theta| exceeds the fp32 error margin derived below;
  (3) the groups inside that margin are the ones that DEFINE theta (the two order statistics the percentile
      interpolates between, and exact ties with them): at most that many distinct GC values per problem.
Margin: GC is K fp32 additions and one division (relative error <= (K + 1) * 2^-24 each side of the sum's
magnitude), theta is one subtraction, one multiplication and one addition on two such values (3 more
roundings), so |GC_fp32 - GC| + |theta_fp32 - theta| <= (2K + 8) * 2^-24 * max|C(tau)|; the margin used is
twice that.  Selection probabilities rel 2e-5.  Also the end of the whole path: sq_score_run's C(tau) fed
straight into sq_score_route on the device."""
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


def check_codes(code, gc32, th32, ref, grp_off, lite, conf, K):
    """The three-way judgement of the routing codes described in the module docstring."""
    per_group = np.diff(grp_off)
    th32_g = np.repeat(th32, per_group)
    is_lite = np.zeros(len(code), dtype=bool) if lite is None else lite.astype(bool)
    undefined = ~is_lite & ~np.isfinite(gc32)
    with np.errstate(invalid="ignore"):
        own = np.where(is_lite, 0, np.where(undefined, 3, np.where(gc32 > th32_g, 1, 2)))     # (1) fp32 compare of the kernel's own outputs
    assert (code == own).all(), np.argwhere(code != own)[:5]
    margin = 2.0 * (2 * K + 8) * 2.0 ** -24 * float(np.nanmax(np.abs(conf))) if len(conf) else 0.0
    th64_g = np.repeat(ref["theta"], per_group)
    with np.errstate(invalid="ignore"):
        far = np.abs(ref["group_fitness"] - th64_g) > margin
    far |= is_lite | undefined | np.isnan(th64_g)                                                 # no comparison is taken there
    assert (code[far] == ref["route"][far]).all(), np.argwhere(far & (code != ref["route"]))[:5]   # (2)
    for q in range(len(per_group)):                                                               # (3)
        near_vals = ref["group_fitness"][grp_off[q]:grp_off[q + 1]][~far[grp_off[q]:grp_off[q + 1]]]
        # the percentile interpolates between two order statistics: at most those two VALUES (and exact ties with
        # them, e.g. groups drawn with the same members) can sit inside the margin
        assert len(np.unique(np.round(near_vals / max(margin, 1e-30)))) <= 3, (q, near_vals)


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
    check_codes(code, out["group_fitness"].cpu().numpy(), th, ref, grp_off, lite, conf, K)
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


def test_route_group_with_an_empty_trajectory():
    """C(tau) of an empty trajectory is NaN: its group takes no part in the percentile and gets code 3 (reading #24);
    the other groups are routed as if it were not there."""
    eng = _eng()
    conf = np.array([6.0, np.nan, 2.0, 4.0, 8.0], dtype=np.float32)
    members = np.array([[0, 2], [1, 3], [3, 4], [2, 3], [1, 1], [0, 4]], dtype=np.int32)
    off = np.array([0, 4, 6], dtype=np.int32)
    lite = np.array([0, 0, 0, 0, 1, 0], dtype=np.uint8)
    out = eng.route(torch.tensor(conf, device=DEV), torch.tensor(members, device=DEV), torch.tensor(off, device=DEV), 50.0,
                    lite_mask=torch.tensor(lite, device=DEV))
    torch.cuda.synchronize()
    ref = O.route(conf, members, off, 50.0, lite)
    assert ref["route"].tolist() == [2, 3, 1, 2, 0, 2]
    assert out["route"].cpu().tolist() == ref["route"].tolist()
    np.testing.assert_array_equal(out["theta"].cpu().numpy(), ref["theta"])          # 4.0 and 7.0: exact in fp32
    gf = out["group_fitness"].cpu().numpy()
    assert np.isnan(gf[1]) and np.isnan(gf[4]) and gf[[0, 2, 3, 5]].tolist() == [4.0, 6.0, 3.0, 7.0]
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
