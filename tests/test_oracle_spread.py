"""Pins for the two extensions of SURVEY 8(f).2 in the oracle (R13, R14; both off by default):
  R13  spread of a cell from its T*N samples (sum f, sum f^2) instead of from T trial values;
  R14  a budget that keeps the flagged cells with the largest spread instead of the first in path order.
Pinned by: direct recomputation from the sample points with numpy, closed-form variances, the
estimator's sampling distribution (z-scores are N(0,1) when the error is a proper 1-sigma), brute-force
top-B selection, and the tree invariants."""
import math

import numpy as np
import pytest

import oracle as O
from paper_1902_07916_b200 import workloads as W
from tests import helpers as H


def _cfg(w, **over):
    return H.oracle_config(w, **over)


def test_unit_sumsq_is_the_sum_of_squared_point_values():
    for w in (W.config1(), W.config2().with_(n_samples=777), W.config3().with_(n_samples=500)):
        cfg = _cfg(w)
        digits = [(w.k - 1) // 2]
        path, coords = O.path_coords(w.dim, w.g, digits)
        x, f = O.unit_points(cfg, 0, path, 1, coords, 2, w.n_samples)
        S, Q = O.unit_sums(cfg, 0, path, 1, coords, 2)
        S0, _ = O.unit_sum(cfg, 0, path, 1, coords, 2)
        assert S == S0                                   # same sequential sum as R5's
        assert abs(Q - float(np.sum(f * f))) <= 1e-13 * float(np.sum(f * f)) + 1e-300
        seq = 0.0
        for v in f:                                      # the stated order: product rounded, then added, sequentially
            seq = seq + float(v) * float(v)
        assert Q == seq


def test_cell_stats_from_samples_match_numpy_and_closed_form():
    w = W.config1()
    cfg = _cfg(w, spread=O.SPREAD_SAMPLES)
    T, N = w.trials, w.n_samples
    for digits in ([0], [21], [63]):
        path, coords = O.path_coords(w.dim, w.g, digits)
        lo, width, V = O.cell_geometry(w.dim, w.lower, w.upper, w.g, 1, coords)
        allf, S, Q = [], [], []
        for t in range(T):
            _, f = O.unit_points(cfg, 0, path, 1, coords, t, N)
            allf.append(f)
            s_, q_ = O.unit_sums(cfg, 0, path, 1, coords, t)
            S.append(s_)
            Q.append(q_)
        allf = np.concatenate(allf)
        mu, s = O.cell_stats_samples(S, Q, V, 1.0, N)
        assert abs(mu - V * allf.mean()) <= 1e-12 * V
        expect = V * math.sqrt(allf.var() / (T * N))     # population variance / M, the standard error of the mean
        assert abs(s - expect) <= 1e-9 * expect
        # closed form of Var f over the cell: the estimate from 10^4 samples is within a few per cent
        var_cf = H.var_sin_sum_box(lo, [a + b for a, b in zip(lo, width)])
        assert abs(s - V * math.sqrt(var_cf / (T * N))) <= 0.05 * s
    # the same numbers come out of the tree driver
    res = O.run(cfg, keep_cells=True)
    l1 = res.levels[0]
    path, coords = O.path_coords(w.dim, w.g, [21])
    S = [O.unit_sums(cfg, 0, path, 1, coords, t) for t in range(T)]
    mu, s = O.cell_stats_samples([a for a, _ in S], [b for _, b in S], 2.5 ** 3, 1.0, N)
    assert l1.mu[21] == mu and l1.s[21] == s
    np.testing.assert_array_equal(l1.Q[21], [b for _, b in S])


def test_constant_integrand_has_zero_spread_and_linear_matches_closed_form():
    w = W.Workload("c", 3, (0.0, 1.0, -1.0), (2.0, 3.0, 1.0), 3, 400, 4, 3, 1.5, 1, W.CONST, W.F64, params=np.array([[0.7]]))
    res = O.run(_cfg(w, spread=O.SPREAD_SAMPLES), keep_cells=True)
    assert np.all(res.levels[0].s == 0.0) and len(res.levels) == 1      # the 2^-40 cut: rounding noise is not a spread
    assert abs(res.value[0] - 0.7 * 8.0) < 1e-12 and res.std[0] == 0.0
    # f = 2 + 3x on [0,1], one cell: Var f = 9/12
    w = W.Workload("l", 1, (0.0,), (1.0,), 1, 20000, 5, 1, 1.5, 3, W.LINEAR, W.F64, params=np.array([[2.0, 3.0]]))
    res = O.run(_cfg(w, spread=O.SPREAD_SAMPLES), keep_cells=True)
    assert abs(res.std[0] - math.sqrt(0.75 / 100000)) <= 0.02 * res.std[0]
    assert abs(res.value[0] - 3.5) <= 4 * res.std[0]


def test_sample_spread_is_a_proper_one_sigma_error():
    """depth 1 stratified MC, 150 seeds: z = (value - closed)/std has mean 0 and variance 1 (with R5/R7's trial spread the
    variance is 1/(T-1) of that, which is why BASELINE.json's 4-sigma gate is loose there)."""
    base = W.Workload("z", 2, (0.0, 0.0), (3.0, 2.0), 3, 60, 4, 1, 1.5, 0, W.SIN_SUM, W.F64)
    closed = H.closed_sin_sum(base.lower, base.upper)
    z = []
    for seed in range(150):
        res = O.run(_cfg(base.with_(seed=1000 + seed), spread=O.SPREAD_SAMPLES))
        z.append((res.value[0] - closed) / res.std[0])
    z = np.array(z)
    assert abs(z.mean()) < 3.5 / math.sqrt(len(z))
    assert 0.72 < z.var() < 1.35


@pytest.mark.parametrize("spread", [O.SPREAD_TRIALS, O.SPREAD_SAMPLES])
def test_largest_spread_budget_is_top_b_by_brute_force(spread):
    w = W.config4(n_instances=3).with_(n_samples=200, depth=3, sigma_multiplier=0.5, max_groups_per_level=3)
    free = O.run(_cfg(w.with_(max_groups_per_level=0, depth=1), spread=spread), keep_cells=True)
    res = O.run(_cfg(w, spread=spread, budget_order=O.BUDGET_LARGEST_SPREAD), keep_cells=True)
    byp = O.run(_cfg(w, spread=spread, budget_order=O.BUDGET_PATH_ORDER), keep_cells=True)
    assert len(res.levels) == 3
    np.testing.assert_array_equal(res.levels[0].s, free.levels[0].s)
    differs = False
    for lev in res.levels[:-1]:
        flagged = lev.s > lev.tau
        for b in range(3):
            idx = np.nonzero(flagged & (lev.instance == b))[0]
            order = sorted(idx, key=lambda i: (-lev.s[i], i))            # brute force: largest s first, ties by position
            want = set(order[:3])
            got = set(np.nonzero(lev.refined.astype(bool) & (lev.instance == b))[0])
            assert got == want
            differs |= want != set(idx[:3])
    assert differs                                   # the case really separates the two orders
    assert any(not np.array_equal(a.refined, b.refined) for a, b in zip(res.levels, byp.levels))
    # invariants: accepted cells tile the domain, accepted means add up to the value
    k = w.k
    for b in range(3):
        tiles = sum(int(np.sum(~lev.refined.astype(bool) & (lev.instance == b))) * k ** (3 - l)
                    for l, lev in enumerate(res.levels, start=1))
        assert tiles == k ** 3
        total = sum(float(np.sum(lev.mu[~lev.refined.astype(bool) & (lev.instance == b)])) for lev in res.levels)
        assert abs(total - res.value[b]) <= 1e-12 * abs(res.value[b])


def test_budget_larger_than_the_flagged_set_changes_nothing():
    w = W.config1().with_(max_groups_per_level=1000)
    a = O.run(_cfg(w, budget_order=O.BUDGET_LARGEST_SPREAD), keep_cells=True)
    b = O.run(_cfg(W.config1()), keep_cells=True)
    assert a.value[0] == b.value[0] and a.std[0] == b.std[0]
    np.testing.assert_array_equal(a.levels[0].refined, b.levels[0].refined)


def test_depth_first_refuses_a_whole_level_budget():
    w = W.config1().with_(max_groups_per_level=2)
    with pytest.raises(ValueError):
        O.run(_cfg(w, traversal=O.DFS, budget_order=O.BUDGET_LARGEST_SPREAD))
