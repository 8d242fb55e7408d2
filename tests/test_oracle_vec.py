"""Pins for the oracle's vector-valued driver (R15, oracle/zmc_oracle_vec.cpp): reduction to the scalar,
independently pinned driver; closed forms; brute-force re-derivation of the "any component" flag rule; invariants.
The user functions are inputs: plain C++ text, the same text NVRTC gets on the CUDA side (tests/vec_sources.py)."""
import numpy as np
import pytest

import oracle as O
from tests import vec_sources as VS


def _cfg(dim=3, g=3, n=400, T=5, depth=2, m=1.0, seed=11, precision=O.F64, lower=None, upper=None, params=None,
         n_instances=1, budget=0, integrand=O.CONST):
    lower = [0.0] * dim if lower is None else lower
    upper = [1.0] * dim if upper is None else upper
    return O.Config(dim=dim, lower=lower, upper=upper, g=g, n_samples=n, trials=T, depth=depth, sigma_multiplier=m,
                    seed=seed, integrand=integrand, precision=precision, params=params, n_instances=n_instances,
                    max_groups_per_level=budget)


# ------------------------------------------------------------ reduction to the scalar driver (C = 1)
@pytest.mark.parametrize("precision", [O.F64, O.F32])
def test_one_component_linear_is_the_scalar_driver_bit_for_bit(precision):
    """A user function that restates LINEAR operation by operation, C = 1: every number of the vector driver
    equals the scalar driver's (which has its own pins) -- sums, (mu, s), tau, refined sets, value, std."""
    p = np.array([[0.3, 1.0, -2.0, 0.5]])
    cfg = _cfg(params=p, precision=precision, integrand=O.LINEAR, lower=[0, -1, 2], upper=[1, 1, 2.5])
    ref = O.run(cfg, keep_cells=True)
    fns = O.compile_user_fn(VS.LINEAR1, "lin1")
    vec = O.run_vec(cfg, 1, fns, keep_cells=True)
    assert len(ref.levels) == len(vec.levels) == 2 and ref.levels[0].n_refined > 0
    for a, b in zip(ref.levels, vec.levels):
        assert (a.n_cells, a.n_refined) == (b.n_cells, b.n_refined)
        assert a.path == b.path
        np.testing.assert_array_equal(a.S, b.S[:, :, 0])
        np.testing.assert_array_equal(a.mu, b.mu[:, 0])
        np.testing.assert_array_equal(a.s, b.s[:, 0])
        np.testing.assert_array_equal(a.tau, b.tau[:, 0])
        np.testing.assert_array_equal(a.refined, b.refined)
    assert ref.value[0] == vec.value[0, 0] and ref.std[0] == vec.std[0, 0]
    assert ref.evals == vec.evals


def test_one_component_sin_f64_is_the_scalar_driver_bit_for_bit():
    cfg = _cfg(integrand=O.SIN_SUM, lower=[0] * 3, upper=[10] * 3, g=4, n=300, m=1.5, seed=1)
    ref = O.run(cfg, keep_cells=True)
    vec = O.run_vec(cfg, 1, O.compile_user_fn(VS.SIN1, "sin1", ("f64",)), keep_cells=True)
    for a, b in zip(ref.levels, vec.levels):
        np.testing.assert_array_equal(a.S, b.S[:, :, 0])
        np.testing.assert_array_equal(a.refined, b.refined)
    assert ref.value[0] == vec.value[0, 0] and ref.std[0] == vec.std[0, 0]


# ------------------------------------------------------------ unit sums = sum of the textbook formulas at the oracle's points
@pytest.mark.parametrize("precision", [O.F64, O.F32])
def test_unit_sums_are_the_formulas_at_the_points(precision):
    cfg = _cfg(precision=precision, lower=[0, 0, -1], upper=[1, 2, 1], n=257, params=np.array([[0.0]]))
    fns = O.compile_user_fn(VS.POLY4, "poly4")
    path, coords = O.path_coords(3, 3, [14])
    S = O.vec_unit_sums(cfg, 4, fns, 0, path, 1, coords, 3)
    x, _ = O.unit_points(cfg, 0, path, 1, coords, 3, 257)       # the scalar oracle's points (pinned against exact rationals)
    want = np.array([(x[:, 0] * x[:, 1]).sum(), (x[:, 2] ** 2).sum(), 3.0 * 257, (x[:, 0] + x[:, 1] * x[:, 2]).sum()])
    np.testing.assert_allclose(S, want, rtol=0, atol=(1e-12 if precision == O.F64 else 3e-5) * 257)
    assert S[2] == 3.0 * 257


# ------------------------------------------------------------ closed forms
def test_polynomial_components_against_closed_forms():
    """f = (x0*x1, x2^2, 3, x0 + x1*x2) over [0,1]x[0,2]x[-1,1]: integrals 2, 4/3, 12, 2."""
    cfg = _cfg(lower=[0, 0, -1], upper=[1, 2, 1], n=2000, depth=2, m=1.0, seed=5)
    r = O.run_vec(cfg, 4, O.compile_user_fn(VS.POLY4, "poly4"))
    closed = np.array([2.0, 4.0 / 3.0, 12.0, 2.0])
    v, s = r.value[0], r.std[0]
    assert abs(v[2] - 12.0) < 1e-12 and s[2] < 1e-14         # a constant component: exact up to the rounding of (sum of T equal values)/T
    for j in (0, 1, 3):
        assert abs(v[j] - closed[j]) < 4 * s[j]
        assert abs(v[j] - closed[j]) < 5 * s[j] / 2.0        # std over-states the error of the mean by ~sqrt(T-1) (R7)
        assert 1e-5 < s[j] < 0.05


# ------------------------------------------------------------ the "any component" rule, by brute force
def test_flag_rule_is_the_union_of_the_components():
    cfg = _cfg(dim=2, g=5, n=300, depth=3, m=1.0, seed=7, lower=[0, 0], upper=[1, 2])
    both = O.run_vec(cfg, 2, O.compile_user_fn(VS.TWO_AXES, "two_axes"), keep_cells=True)
    only0 = O.run_vec(cfg, 1, O.compile_user_fn(VS.AXIS0, "axis0"), keep_cells=True)
    only1 = O.run_vec(cfg, 1, O.compile_user_fn(VS.AXIS1, "axis1"), keep_cells=True)
    k = 25
    l1 = both.levels[0]
    # level 1 is the same 25 cells with the same streams in all three runs
    np.testing.assert_array_equal(l1.s[:, 0], only0.levels[0].s[:, 0])
    np.testing.assert_array_equal(l1.s[:, 1], only1.levels[0].s[:, 0])
    union = (only0.levels[0].refined | only1.levels[0].refined)
    assert only0.levels[0].refined.sum() > 0 and only1.levels[0].refined.sum() > 0
    assert (only0.levels[0].refined != only1.levels[0].refined).any()
    np.testing.assert_array_equal(l1.refined, union)
    # every level: tau and flags re-derived in numpy from the dumped (mu, s)
    for lev, L in enumerate(both.levels, start=1):
        G = L.n_cells // k
        sg = L.s.reshape(G, k, 2)
        mean = sg.mean(axis=1)
        pstd = np.sqrt(((sg - mean[:, None, :]) ** 2).mean(axis=1))
        tau = mean + 1.0 * pstd
        np.testing.assert_allclose(L.tau.reshape(G, k, 2)[:, 0, :], tau, rtol=1e-13, atol=1e-300)
        flag = (sg > L.tau.reshape(G, k, 2)).any(axis=2).reshape(-1) & (lev < 3)
        np.testing.assert_array_equal(L.refined.astype(bool), flag)
    # the next level holds exactly the children of the refined cells, in path order
    for a, b in zip(both.levels[:-1], both.levels[1:]):
        parents = [p for p, r in zip(a.path, a.refined) if r]
        assert b.path == [p * k + j for p in parents for j in range(k)]
    # invariants: accepted cells tile the domain; accepted means add up to the value
    Lmax = 3
    assert sum((L.n_cells - L.n_refined) * k ** (Lmax - lev) for lev, L in enumerate(both.levels, start=1)) == k ** Lmax
    for j in range(2):
        acc = sum(L.mu[~L.refined.astype(bool), j].sum() for L in both.levels)
        assert abs(acc - both.value[0, j]) < 1e-12
        accv = sum((L.s[~L.refined.astype(bool), j] ** 2).sum() for L in both.levels)
        assert abs(np.sqrt(accv) - both.std[0, j]) < 1e-12


def test_duplicate_component_changes_nothing():
    cfg = _cfg(dim=2, g=5, n=300, depth=2, m=1.0, seed=7, lower=[0, 0], upper=[1, 2])
    one = O.run_vec(cfg, 1, O.compile_user_fn(VS.AXIS0, "axis0"), keep_cells=True)
    two = O.run_vec(cfg, 2, O.compile_user_fn(VS.AXIS0_TWICE, "axis0_twice"), keep_cells=True)
    for a, b in zip(one.levels, two.levels):
        np.testing.assert_array_equal(a.refined, b.refined)
        np.testing.assert_array_equal(b.mu[:, 0], b.mu[:, 1])
        np.testing.assert_array_equal(a.mu[:, 0], b.mu[:, 0])
    assert one.value[0, 0] == two.value[0, 0] == two.value[0, 1]
    assert one.std[0, 0] == two.std[0, 1]


def test_budget_keeps_the_first_flagged_cells_in_path_order_per_instance():
    p = np.array([[1.0], [2.5]])
    free = O.run_vec(_cfg(dim=2, g=5, n=300, depth=2, seed=9, params=p, n_instances=2), 2,
                     O.compile_user_fn(VS.SCALED_AXES, "scaled_axes"), keep_cells=True)
    cut = O.run_vec(_cfg(dim=2, g=5, n=300, depth=2, seed=9, params=p, n_instances=2, budget=2), 2,
                    O.compile_user_fn(VS.SCALED_AXES, "scaled_axes"), keep_cells=True)
    f1, c1 = free.levels[0], cut.levels[0]
    np.testing.assert_array_equal(f1.s, c1.s)
    for b in (0, 1):
        flagged = np.nonzero(f1.refined.astype(bool) & (f1.instance == b))[0]
        assert len(flagged) > 2
        kept = np.nonzero(c1.refined.astype(bool) & (c1.instance == b))[0]
        np.testing.assert_array_equal(kept, flagged[:2])
    assert c1.n_truncated == f1.n_refined - 4 and cut.levels[1].n_cells == 4 * 25
    # instances are independent: instance 1 sees its own parameter (values scale with p)
    assert abs(free.value[1, 0] / free.value[0, 0] - 2.5) < 0.2


def test_vector_driver_rejects_what_it_does_not_define():
    cfg = _cfg()
    fns = O.compile_user_fn(VS.POLY4, "poly4")
    with pytest.raises(ValueError):
        O.run_vec(cfg, 0, fns)
    cfg.budget_order = O.BUDGET_LARGEST_SPREAD
    with pytest.raises(ValueError):
        O.run_vec(cfg, 4, fns)


# ------------------------------------------------------------ R13 per component (spread from the samples)
@pytest.mark.parametrize("precision", [O.F64, O.F32])
def test_spread_from_samples_one_component_is_the_scalar_driver_bit_for_bit(precision):
    p = np.array([[0.3, 1.0, -2.0, 0.5]])
    cfg = _cfg(params=p, precision=precision, integrand=O.LINEAR, lower=[0, -1, 2], upper=[1, 1, 2.5], m=0.5)
    cfg.spread = O.SPREAD_SAMPLES
    ref = O.run(cfg, keep_cells=True)
    vec = O.run_vec(cfg, 1, O.compile_user_fn(VS.LINEAR1, "lin1"), keep_cells=True)
    assert len(ref.levels) == len(vec.levels) and ref.levels[0].n_refined > 0
    for a, b in zip(ref.levels, vec.levels):
        np.testing.assert_array_equal(a.S, b.S[:, :, 0])
        np.testing.assert_array_equal(a.Q, b.Q[:, :, 0])
        np.testing.assert_array_equal(a.mu, b.mu[:, 0])
        np.testing.assert_array_equal(a.s, b.s[:, 0])
        np.testing.assert_array_equal(a.tau, b.tau[:, 0])
        np.testing.assert_array_equal(a.refined, b.refined)
    assert ref.value[0] == vec.value[0, 0] and ref.std[0] == vec.std[0, 0]


def test_spread_from_samples_per_component_against_numpy():
    """Every component's cell spread = V * sqrt(var(f_j over the cell's T*N samples) / (T*N)), recomputed with numpy from the
    scalar oracle's points; sums of squares = the formulas squared at those points; a constant component has spread exactly 0."""
    cfg = _cfg(lower=[0, 0, -1], upper=[1, 2, 1], n=300, T=4, depth=1, params=np.array([[0.0]]))
    cfg.spread = O.SPREAD_SAMPLES
    fns = O.compile_user_fn(VS.POLY4, "poly4")
    r = O.run_vec(cfg, 4, fns, keep_cells=True)
    L1 = r.levels[0]
    V = (1.0 / 3) * (2.0 / 3) * (2.0 / 3)
    for cell in (0, 13, 26):
        path, coords = O.path_coords(3, 3, [cell])
        vals = []
        for t in range(4):
            x, _ = O.unit_points(cfg, 0, path, 1, coords, t, 300)
            f = np.stack([x[:, 0] * x[:, 1], x[:, 2] ** 2, np.full(300, 3.0), x[:, 0] + x[:, 1] * x[:, 2]], axis=1)
            vals.append(f)
            S, Q = O.vec_unit_sums_sq(cfg, 4, fns, 0, path, 1, coords, t)
            np.testing.assert_allclose(S, f.sum(axis=0), rtol=1e-13)
            np.testing.assert_allclose(Q, (f * f).sum(axis=0), rtol=1e-13)
            np.testing.assert_allclose(L1.Q[cell, t], Q, rtol=0, atol=0)
        allf = np.concatenate(vals, axis=0)
        want = V * np.sqrt(allf.var(axis=0) / allf.shape[0])
        np.testing.assert_allclose(L1.s[cell, [0, 1, 3]], want[[0, 1, 3]], rtol=1e-9)
        assert L1.s[cell, 2] == 0.0
    assert r.std[0, 2] == 0.0


def test_spread_from_samples_gives_a_one_sigma_error_per_component():
    """z = (value - closed form) / std over seeds: mean ~ 0 and variance ~ 1 for every non-constant component (R13's claim)."""
    closed = np.array([2.0, 4.0 / 3.0, 12.0, 2.0])
    fns = O.compile_user_fn(VS.POLY4, "poly4")
    z = []
    for seed in range(60):
        cfg = _cfg(lower=[0, 0, -1], upper=[1, 2, 1], n=60, T=2, depth=1, seed=1000 + seed, g=2)
        cfg.spread = O.SPREAD_SAMPLES
        r = O.run_vec(cfg, 4, fns)
        z.append((r.value[0, [0, 1, 3]] - closed[[0, 1, 3]]) / r.std[0, [0, 1, 3]])
    z = np.array(z)
    assert np.all(np.abs(z.mean(axis=0)) < 0.45)
    assert np.all((z.var(axis=0) > 0.55) & (z.var(axis=0) < 1.6))
