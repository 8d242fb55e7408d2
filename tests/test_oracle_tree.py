"""Pins for the oracle's statistics and tree driver (R5-R7, R11, R12): a worked example from an
independent prototype, hand-computed cases, closed forms, brute-force quadrature, invariants and
the estimator's sampling distribution."""
import math
import os

import numpy as np
import pytest
from scipy import integrate

import oracle as O
from paper_1902_07916_b200 import workloads as W
from tests import helpers as H

GOLD = os.path.join(os.path.dirname(__file__), "golden", "config1_worked.txt")


def _gold():
    g = {}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        g.setdefault(k, []).append(v)
    return g


@pytest.fixture(scope="module")
def run1():
    return O.run(H.oracle_config(W.config1()), keep_cells=True)


# ------------------------------------------------------------ worked example (config 1)
def test_config1_worked_example(run1):
    g = _gold()
    cfg = H.oracle_config(W.config1())
    x, f = O.unit_points(cfg, 0, 0, 1, [0, 0, 0], 0, 1)
    assert list(x[0]) == [float(v) for v in g["point0"][0]]
    assert abs(f[0] - float(g["f0"][0][0])) < 1e-15
    l1, l2 = run1.levels
    V = 2.5**3
    trials = [float(v) for v in g["cell0_trials"][0]]
    np.testing.assert_allclose(l1.S[0] * V / 2000, trials, rtol=2e-10)
    for c, mu, s in g["cell"]:
        assert abs(l1.mu[int(c)] - float(mu)) < 2e-9 and abs(l1.s[int(c)] - float(s)) < 2e-9
    assert abs(l1.tau[0] - float(g["tau1"][0][0])) < 2e-10
    assert list(np.nonzero(l1.refined)[0]) == [int(v) for v in g["refined1"][0]]
    assert (l1.n_cells, l1.n_refined, l2.n_cells, l2.n_refined) == (64, 5, 320, 0)
    for parent, tau in g["tau2"]:
        idx = [i for i, p in enumerate(l2.path) if p // 64 == int(parent)]
        assert len(idx) == 64 and abs(l2.tau[idx[0]] - float(tau)) < 2e-12
    assert abs(run1.value[0] - float(g["value"][0][0])) < 2e-9
    assert abs(run1.std[0] - float(g["std"][0][0])) < 2e-9
    # within 4 sigma of the closed form (BASELINE.json)
    closed = H.closed_sin_sum([0] * 3, [10] * 3)
    assert abs(closed - (-4.587209322781949)) < 1e-13
    assert abs(run1.value[0] - closed) < 4 * run1.std[0]


# ------------------------------------------------------------ hand-computed statistics
def test_cell_stats_hand_case():
    I, mu, s = O.cell_stats([1, 2, 3, 4, 5], volume=2.0, prefactor=1.0, n_samples=10)
    np.testing.assert_allclose(I, [0.2, 0.4, 0.6, 0.8, 1.0], rtol=1e-15)
    assert abs(mu - 0.6) < 1e-15 and abs(s - 0.2 * math.sqrt(2.0)) < 1e-15   # ddof 0
    _, mu2, s2 = O.cell_stats([1, 2, 3, 4, 5], 2.0, 3.0, 10)
    assert abs(mu2 - 1.8) < 1e-15 and abs(s2 - 0.6 * math.sqrt(2.0)) < 1e-15
    _, mu1, s1 = O.cell_stats([7.0], 1.0, 1.0, 7)
    assert (mu1, s1) == (1.0, 0.0)                                            # T = 1 -> s = 0


def test_threshold_hand_case():
    s = [1.0, 2.0, 3.0, 10.0]                       # mean 4, population variance 12.5
    assert abs(O.threshold(s, 1.0) - (4 + math.sqrt(12.5))) < 1e-15
    assert abs(O.threshold(s, 0.0) - 4.0) < 1e-15
    assert abs(O.threshold(s, 5.0) - (4 + 5 * math.sqrt(12.5))) < 1e-14
    assert O.threshold([0.3] * 7, 1.5) == 0.3       # all equal -> tau = s -> nothing is "larger than"
    assert O.threshold([0.0] * 7, 1.5) == 0.0


# ------------------------------------------------------------ closed forms pinned by brute-force quadrature
def test_closed_forms_by_quadrature_1d_2d():
    v1, _ = integrate.quad(np.sin, 0, 10, epsabs=1e-13)
    assert abs(H.closed_sin_sum([0], [10]) - v1) < 1e-11
    v2, _ = integrate.dblquad(lambda y, x: np.sin(x + y), 0, 10, 0, 10, epsabs=1e-11)
    assert abs(H.closed_sin_sum([0, 0], [10, 10]) - v2) < 1e-9
    p = [2.0, 30.0, 0.3, 0.6]
    g1, _ = integrate.quad(lambda x: p[0] * np.exp(-p[1] * (x - p[2]) ** 2), 0, 1, epsabs=1e-13)
    assert abs(H.closed_exp_quad(p[:3], [0], [1]) - g1) < 1e-11
    g2, _ = integrate.dblquad(lambda y, x: p[0] * np.exp(-p[1] * ((x - p[2]) ** 2 + (y - p[3]) ** 2)), 0, 1, 0, 1, epsabs=1e-11)
    assert abs(H.closed_exp_quad(p, [0, 0], [1, 1]) - g2) < 1e-9
    assert abs(H.closed_sin_sum([0] * 6, [10] * 6) - (-49.16507381641946)) < 1e-12
    assert abs(H.closed_exp_quad(W.gaussian_params(9, 0.01)[0], [-1] * 9, [1] * 9) - 1.0) < 1e-12


@pytest.mark.parametrize("prec", [O.F64, O.F32])
def test_integrand_values_at_points(prec):
    """f returned by the oracle equals the textbook formula evaluated (numpy, FP64) at the returned x."""
    tol = 1e-14 if prec == O.F64 else 4e-6
    cfg = O.Config(4, [0, 1, -2, 0.5], [10, 3, 2, 0.75], 3, 64, 2, 1, 1.5, 11, O.SIN_SUM, prec)
    P, cc = O.path_coords(4, 3, [50])
    x, f = O.unit_points(cfg, 0, P, 1, cc, 1, 64)
    np.testing.assert_allclose(f, np.sin(x.sum(1)), atol=tol)
    params = np.array([[1.0, 7.5, 0.3, 0.5, 0.7, 0.2]])
    cfg = O.Config(4, [0] * 4, [1] * 4, 2, 64, 2, 1, 1.5, 11, O.EXP_QUAD, prec, params=params)
    P, cc = O.path_coords(4, 2, [9])
    x, f = O.unit_points(cfg, 0, P, 1, cc, 0, 64)
    y = x if prec == O.F32 else x - params[0, 2:]      # FP32 path returns x - c (R8)
    np.testing.assert_allclose(f, np.exp(-7.5 * (y**2).sum(1)), rtol=max(tol, 1e-13))
    lin = np.array([[0.5, 1.0, -2.0, 3.0, 0.25]])
    cfg = O.Config(4, [0] * 4, [1] * 4, 2, 64, 2, 1, 1.5, 11, O.LINEAR, prec, params=lin)
    x, f = O.unit_points(cfg, 0, P, 1, cc, 0, 64)
    np.testing.assert_allclose(f, 0.5 + x @ lin[0, 1:], rtol=1e-6 if prec == O.F32 else 1e-14)


def test_unit_sum_is_sum_of_point_values():
    cfg = O.Config(3, [0] * 3, [10] * 3, 4, 777, 3, 2, 1.5, 5, O.SIN_SUM, O.F32)   # ragged: 777*3 words, not a multiple of 4
    P, cc = O.path_coords(3, 4, [13, 40])
    S, Sabs = O.unit_sum(cfg, 0, P, 2, cc, 2)
    _, f = O.unit_points(cfg, 0, P, 2, cc, 2, 777)
    assert abs(S - f.sum()) < 1e-12 and abs(Sabs - np.abs(f).sum()) < 1e-12
    # samples really are consecutive words of the flat stream: sample s, dim d <- word s*D+d
    words = O.unit_words(5, 0, P, 2, 2, 0, 777 * 3)
    lo, w, _ = O.cell_geometry(3, [0] * 3, [10] * 3, 4, 2, cc)
    x, _ = O.unit_points(cfg, 0, P, 2, cc, 2, 777)
    for s in (0, 1, 2, 3, 776):
        for d in range(3):
            assert x[s, d] == float(O.map_f32(int(words[s * 3 + d]), lo[d], w[d]))


# ------------------------------------------------------------ special cases with textbook answers
def test_const_and_linear_integrands():
    c = O.Config(3, [0, 1, 2], [2, 4, 3], 3, 50, 4, 2, 1.5, 3, O.CONST, O.F64, params=np.array([[2.5]]))
    r = O.run(c)
    assert abs(r.value[0] - 2.5 * 6.0) < 1e-13 and r.std[0] < 1e-14
    assert r.levels[0].n_refined == 0            # all s equal (zero) -> nothing flagged (R7 degenerate case)
    lin = np.array([[0.5, 1.0, -2.0, 3.0]])
    for prec in (O.F64, O.F32):
        c = O.Config(3, [0, 1, 2], [2, 4, 3], 3, 400, 5, 1, 1.5, 3, O.LINEAR, prec, params=lin)
        r = O.run(c)
        closed = H.closed_linear(lin[0], [0, 1, 2], [2, 4, 3])
        assert abs(r.value[0] - closed) < 4 * r.std[0] / 2 + 1e-12


def test_plain_mc_special_case_g1_depth1():
    """g = 1, L = 1 is textbook plain MC: sigma of one trial = Vol * sqrt(Var f / N); never refines."""
    lower, upper = [0.0, 0.0], [3.0, 2.0]
    T, N = 200, 500
    c = O.Config(2, lower, upper, 1, N, T, 1, 1.5, 17, O.SIN_SUM, O.F64)
    r = O.run(c, keep_cells=True)
    assert r.levels[0].n_cells == 1 and r.levels[0].n_refined == 0
    sigma = 6.0 * math.sqrt(H.var_sin_sum_box(lower, upper) / N)
    assert abs(r.std[0] / sigma - 1) < 4 / math.sqrt(2 * T)          # s over T=200 trials estimates sigma
    assert abs(r.value[0] - H.closed_sin_sum(lower, upper)) < 4 * sigma / math.sqrt(T)


def test_depth1_stratified_variance_and_unbiasedness():
    """Depth 1 = plain stratified MC. Over R seeds: z = (value - closed)/(std/sqrt(T-1)) has mean ~ 0 and
    variance ~ 1 (ddof 0, quadrature collection, no sqrt(T): R5/R7), and E[std^2] = (T-1)/T sum_c V_c^2 Var_c f / N."""
    dim, g, N, T, R = 3, 3, 300, 5, 60
    lower, upper = [0.0] * dim, [10.0] * dim
    closed = H.closed_sin_sum(lower, upper)
    w = 10.0 / g
    pred = 0.0
    for i in range(g):
        for j in range(g):
            for l in range(g):
                lo = [i * w, j * w, l * w]
                pred += (w**dim) ** 2 * H.var_sin_sum_box(lo, [v + w for v in lo]) / N
    pred *= (T - 1) / T
    z, v = [], []
    for seed in range(100, 100 + R):
        r = O.run(O.Config(dim, lower, upper, g, N, T, 1, 1.5, seed, O.SIN_SUM, O.F64))
        z.append((r.value[0] - closed) / (r.std[0] / math.sqrt(T - 1)))
        v.append(r.std[0] ** 2)
    z = np.array(z)
    assert abs(z.mean()) < 4 / math.sqrt(R)
    assert 0.55 < z.var() < 1.7
    assert abs(np.mean(v) / pred - 1) < 0.08


# ------------------------------------------------------------ tree invariants
def _check_tiling(res, k, L, n_inst=1):
    total = 0
    for lev, rec in enumerate(res.levels, start=1):
        total += (rec.n_cells - rec.n_refined) * k ** (L - lev)
    assert total == n_inst * k**L


def test_tree_invariants_and_traversal_independence(run1):
    w = W.config1()
    k, L = w.k, w.depth
    _check_tiling(run1, k, L)
    acc_mu = sum(float(rec.mu[rec.refined == 0].sum()) for rec in run1.levels)
    acc_var = sum(float((rec.s[rec.refined == 0] ** 2).sum()) for rec in run1.levels)
    assert abs(acc_mu - run1.value[0]) < 1e-12 and abs(math.sqrt(acc_var) - run1.std[0]) < 1e-12
    assert run1.evals == sum(rec.n_cells for rec in run1.levels) * w.trials * w.n_samples
    # level-2 cells are exactly the children of the refined level-1 cells, in ascending path order
    l1, l2 = run1.levels
    parents = [p for p, r in zip(l1.path, l1.refined) if r]
    assert l2.path == [p * k + j for p in parents for j in range(k)]
    # flags follow the strict rule s > tau
    assert np.array_equal(l1.refined.astype(bool), l1.s > l1.tau)
    assert not l2.refined.any()                       # level L is never refined
    # depth-first recursion (the paper's Fig. 1) gives the same numbers (R2)
    rd = O.run(H.oracle_config(w, traversal=O.DFS))
    assert abs(rd.value[0] - run1.value[0]) < 1e-13 and abs(rd.std[0] - run1.std[0]) < 1e-13
    assert [(a.n_cells, a.n_refined) for a in rd.levels] == [(a.n_cells, a.n_refined) for a in run1.levels]


def test_depth_semantics_and_monotone_in_m():
    w = W.config1()
    r1 = O.run(H.oracle_config(w.with_(depth=1)), keep_cells=True)      # depth 1: one partition, nothing refined
    assert len(r1.levels) == 1 and r1.levels[0].n_refined == 0 and r1.levels[0].n_cells == 64
    prev = None
    for m in (0.0, 0.5, 1.5, 3.0, 50.0):
        r = O.run(H.oracle_config(w.with_(sigma_multiplier=m)), keep_cells=True)
        flagged = set(np.nonzero(r.levels[0].refined)[0])
        if prev is not None:
            assert flagged <= prev
        prev = flagged
        _check_tiling(r, w.k, w.depth)
    assert prev == set()                                               # huge m: never refines, run ends at level 1
    assert len(r.levels) == 1


def test_budget_first_B_in_path_order():
    w = W.config1().with_(depth=3, sigma_multiplier=0.5, n_samples=200)
    full = O.run(H.oracle_config(w), keep_cells=True)
    B = 3
    cut = O.run(H.oracle_config(w.with_(max_groups_per_level=B)), keep_cells=True)
    f1 = list(np.nonzero(full.levels[0].refined)[0])
    assert len(f1) > B
    assert list(np.nonzero(cut.levels[0].refined)[0]) == f1[:B]         # first B flagged cells in ascending path order
    assert cut.levels[0].n_truncated == len(f1) - B
    for rec in cut.levels:
        assert rec.n_refined <= B
    _check_tiling(cut, w.k, w.depth)
    dfs = O.run(H.oracle_config(w.with_(max_groups_per_level=B), traversal=O.DFS))
    assert abs(dfs.value[0] - cut.value[0]) < 1e-12 and abs(dfs.std[0] - cut.std[0]) < 1e-12


def test_pooled_scope_option():
    w = W.config1().with_(depth=3, sigma_multiplier=0.5, n_samples=200)
    grp = O.run(H.oracle_config(w), keep_cells=True)
    pool = O.run(H.oracle_config(w, threshold_scope=O.SCOPE_POOLED), keep_cells=True)
    assert np.array_equal(grp.levels[0].refined, pool.levels[0].refined)     # one group at level 1: same
    l2 = pool.levels[1]
    assert len(set(l2.tau)) == 1 and abs(l2.tau[0] - O.threshold(l2.s, 0.5)) < 1e-15
    assert len(set(grp.levels[1].tau)) == grp.levels[0].n_refined


def test_batched_instances_are_independent_runs():
    p = W.batched_params(3, 2, seed=9)
    base = dict(dim=2, lower=[0, 0], upper=[1, 1], g=3, n_samples=300, trials=5, depth=2, sigma_multiplier=1.0,
                seed=4, integrand=O.EXP_QUAD, precision=O.F32)
    rb = O.run(O.Config(**base, params=p, n_instances=3), keep_cells=True)
    r0 = O.run(O.Config(**base, params=p[:1], n_instances=1))
    assert rb.value[0] == r0.value[0] and rb.std[0] == r0.std[0]         # instance 0 uses Kd(seed, 0)
    same = O.run(O.Config(**base, params=np.repeat(p[:1], 2, 0), n_instances=2))
    assert same.value[0] != same.value[1]                                # same function, different stream
    for b in range(3):
        closed = H.closed_exp_quad(p[b], [0, 0], [1, 1])
        assert abs(rb.value[b] - closed) < 4 * rb.std[b]
    _check_tiling(rb, 9, 2, n_inst=3)
    l2 = rb.levels[1]
    assert list(l2.instance) == sorted(l2.instance)                      # lists stay grouped by instance


def test_narrow_gaussian_tree_homes_in_fp32_extended_range():
    """A reduced config 3 (3-D, sigma = 0.01): FP32 evaluation would underflow at level 1 (finding F2);
    with zexp assembled in FP64 range (R9) the centre cell is flagged at every level and the result is 1."""
    w = W.config3()
    small = w.with_(dim=3, lower=(-1.0,) * 3, upper=(1.0,) * 3, n_samples=4000, params=W.gaussian_params(3, 0.01), seed=3)
    r = O.run(H.oracle_config(small), keep_cells=True)
    centre = (27 - 1) // 2
    for lev in range(3):
        assert list(np.nonzero(r.levels[lev].refined)[0]) == [centre]
    assert abs(r.value[0] - 1.0) < 4 * r.std[0] and r.std[0] < 0.05
    r64 = O.run(H.oracle_config(small, precision=O.F64))
    assert abs(r64.value[0] - 1.0) < 4 * r64.std[0]


def test_fanned_out_driver_is_the_oracle_bit_for_bit():
    """tests/whole_tree.oracle_tree_fanned (per-unit sums in a process pool, then orc_cell_stats / orc_threshold level by level) is what the
    GPU suite uses for BASELINE.json configs[2] whole; here it is pinned to oracle.run on small trees: every number the same bits."""
    from tests import whole_tree as WT
    for w in (W.config1(), W.config3().with_(g=2, n_samples=40, depth=3, sigma_multiplier=0.5),
              W.Workload("s2", 2, (0.0, 0.0), (7.0, 5.0), 5, 64, 5, 4, 0.3, 9, W.SIN_SUM, W.F32)):
        a = O.run(H.oracle_config(w), keep_cells=True)
        b = WT.oracle_tree_fanned(w, processes=2, cells_per_job=7)
        assert len(a.levels) == len(b.levels) and a.evals == b.evals
        for la, lb in zip(a.levels, b.levels):
            assert (la.n_cells, la.n_refined) == (lb.n_cells, lb.n_refined) and la.path == lb.path
            for f in ("instance", "S", "mu", "s", "tau", "refined"):
                np.testing.assert_array_equal(getattr(la, f), getattr(lb, f), err_msg=f)
        assert abs(a.value[0] - b.value[0]) <= 1e-13 * max(abs(a.value[0]), a.std[0]) and abs(a.std[0] - b.std[0]) <= 1e-13 * a.std[0]
