"""Pins for the routing row of the oracle: GC(g) (Eq. 4 right,
PAPER.md:160), the per-problem percentile threshold (Eq. 6), the model assignment
(Eq. 7 / "easy means GC(g) > theta_q") and the fitness-weighted selection
probabilities.  CPU only."""
import math

import numpy as np
import pytest

from oracle import sq_oracle as O


def test_group_confidence_hand_values():
    c = [1.0, 2.0, 4.0, 8.0, 16.0]
    gm = [[0, 1, 2, 3], [4, 4, 4, 4], [3, 0, 1, 4]]
    assert O.group_confidence(c, gm).tolist() == [3.75, 16.0, 6.75]
    assert O.group_confidence(c, [[2]]).tolist() == [4.0]                      # K = 1: GC = C


def test_percentile_special_cases():
    v = [5.0, 1.0, 3.0, 2.0, 4.0]
    assert O.percentile_threshold(v, 0) == 1.0                                  # p = 0 -> min
    assert O.percentile_threshold(v, 100) == 5.0                                # p = 100 -> max
    assert O.percentile_threshold(v, 50) == 3.0                                 # odd n -> median
    assert O.percentile_threshold([1.0, 2.0], 50) == 1.5                        # even n -> midpoint
    assert O.percentile_threshold([7.0], 37) == 7.0
    assert math.isnan(O.percentile_threshold([], 50))
    assert O.percentile_threshold([0.0, 10.0], 25) == 2.5                       # linear interpolation
    assert O.percentile_threshold(v, 30) == pytest.approx(1.0 + 0.3 * 4)        # rank 1.2 -> 2.2


def test_percentile_matches_library_routine():
    rng = np.random.default_rng(0)
    for n in (1, 2, 3, 16, 17, 200):
        v = rng.normal(size=n)
        for p in (0, 10, 33.3, 50, 75, 99, 100):
            assert O.percentile_threshold(v, p) == pytest.approx(np.percentile(v, p), abs=1e-13)


def test_percentile_is_monotone_and_bounded():
    rng = np.random.default_rng(1)
    v = rng.uniform(3, 9, size=31)
    th = [O.percentile_threshold(v, p) for p in range(0, 101, 5)]
    assert all(a <= b for a, b in zip(th, th[1:]))
    assert th[0] == v.min() and th[-1] == v.max()


def test_route_hand_example():
    # two problems; problem 0 has 4 groups, problem 1 has 3 groups of which one is lite
    c = np.array([6.0, 6.0, 2.0, 2.0, 4.0, 4.0, 9.0, 1.0, 5.0, 5.0, 5.0, 7.0])
    gm = [[0, 1], [2, 3], [4, 5], [6, 7],          # GC = 6, 2, 4, 5
          [8, 9], [10, 11], [0, 2]]                # GC = 5, 6, 4
    off = [0, 4, 7]
    lite = [0, 0, 0, 0, 0, 0, 1]
    r = O.route(c, gm, off, 50.0, lite)
    assert r["group_fitness"].tolist() == [6, 2, 4, 5, 5, 6, 4]
    assert r["theta"].tolist() == [4.5, 5.5]       # median of {6,2,4,5}; of the non-lite {5,6}
    assert r["route"].tolist() == [1, 2, 2, 1, 2, 1, 0]     # GC > theta -> Model 1; lite stays 0
    # strict ">": a group exactly at the threshold goes to Model 2
    r2 = O.route([3.0, 3.0, 3.0], [[0], [1], [2]], [0, 3], 50.0)
    assert r2["theta"][0] == 3.0 and r2["route"].tolist() == [2, 2, 2]
    # all groups lite -> NaN threshold, nothing routed
    r3 = O.route([1.0, 2.0], [[0], [1]], [0, 2], 50.0, [1, 1])
    assert math.isnan(r3["theta"][0]) and r3["route"].tolist() == [0, 0]


def test_routing_fraction_tracks_the_percentile():
    # "the routing fraction remains approximately p/100 regardless" of the problem's difficulty
    rng = np.random.default_rng(2)
    Q, M, K = 50, 64, 4
    c = rng.normal(size=Q * 16) + np.repeat(rng.normal(scale=5, size=Q), 16)   # per-problem difficulty shift
    gm = np.concatenate([rng.integers(0, 16, size=(M, K)) + 16 * q for q in range(Q)])
    off = np.arange(0, Q * M + 1, M)
    for p in (20, 50, 80):
        r = O.route(c, gm, off, float(p))
        frac_m2 = (r["route"] == 2).mean()
        assert abs(frac_m2 - p / 100) < 0.03
    # shifting a problem's confidences shifts its theta and leaves its routing unchanged
    r0 = O.route(c[:16], gm[:M], [0, M], 40.0)
    r1 = O.route(c[:16] + 100.0, gm[:M], [0, M], 40.0)
    assert (r0["route"] == r1["route"]).all() and r1["theta"][0] == pytest.approx(r0["theta"][0] + 100.0)


def test_group_with_an_empty_trajectory_is_left_out_of_the_percentile():
    # C(tau) of an empty trajectory is NaN (reading #9); its group has no fitness: code 3, and theta is the
    # percentile of the remaining groups (reading #24)
    c = np.array([6.0, np.nan, 2.0, 4.0, 8.0])
    gm = [[0, 2], [1, 3], [3, 4], [2, 3]]          # GC = 4, NaN, 6, 3
    r = O.route(c, gm, [0, 4], 50.0)
    assert np.isnan(r["group_fitness"][1]) and r["group_fitness"][[0, 2, 3]].tolist() == [4.0, 6.0, 3.0]
    assert r["theta"][0] == 4.0                    # median of {4, 6, 3}
    assert r["route"].tolist() == [2, 3, 1, 2]
    same = O.route(c[[0, 2, 3, 4]], [[0, 1], [2, 3], [1, 2]], [0, 3], 50.0)       # the problem without that group
    assert same["theta"][0] == r["theta"][0] and same["route"].tolist() == [2, 1, 2]
    # a lite group stays lite even if its fitness is undefined; only undefined groups -> NaN threshold
    r2 = O.route(c, [[1, 1], [1, 0]], [0, 2], 50.0, [1, 0])
    assert r2["route"].tolist() == [0, 3] and math.isnan(r2["theta"][0])


def test_selection_probabilities():
    f = [1.0, 2.0, 3.0, 10.0, 10.0]
    off = [0, 3, 5]
    pr = O.selection_probabilities(f, off, 0.5)
    assert pr[:3].sum() == pytest.approx(1.0) and pr[3:].sum() == pytest.approx(1.0)
    assert pr[3] == pr[4] == 0.5
    z = math.exp(2) + math.exp(4) + math.exp(6)
    np.testing.assert_allclose(pr[:3], [math.exp(2) / z, math.exp(4) / z, math.exp(6) / z], rtol=1e-13)
    # two candidates: logistic in the fitness gap; zeta -> infinity: uniform
    p2 = O.selection_probabilities([0.0, 1.0], [0, 2], 0.5)
    assert p2[1] == pytest.approx(1 / (1 + math.exp(-2.0)))
    assert O.selection_probabilities([3.0, 9.0, -4.0], [0, 3], 1e12).tolist() == pytest.approx([1 / 3] * 3)
    assert O.selection_probabilities([5.0, 700.0], [0, 2], 0.5)[1] == pytest.approx(1.0)   # no overflow
