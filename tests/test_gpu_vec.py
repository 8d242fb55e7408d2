"""GPU parity of vector-valued user integrands (R15) against oracle/zmc_oracle_vec.cpp, through the C ABI:
whole trees cell by cell (sums, per-component mu/s/tau, refined sets, results), sibling groups of several control tiles,
chunked units, instances with budgets, a 6-D eight-component case with sampled units + a numpy re-derivation of the control path,
and the API's error states. The user functions are the same text on both sides (tests/vec_sources.py)."""
import numpy as np
import pytest

import oracle as O
from paper_1902_07916_b200 import binding as B
from tests import vec_sources as VS

pytestmark = pytest.mark.gpu


def _make(dim, lower, upper, g, n, T, depth, m, seed, src, fn, C, precision, params=None, n_instances=1, budget=0, cap=1 << 16, opts=None):
    it = B.Integrator(dim, lower, upper, g, n, T, depth, m, seed)
    it.set_option(B.OPT_PRECISION, B.F32 if precision == O.F32 else B.F64)
    it.set_integrand_source_vec(src, fn, C, params, n_instances)
    it.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
    it.set_option(B.OPT_MAX_CELLS_PER_LEVEL, cap)
    if budget:
        it.set_option(B.OPT_MAX_GROUPS_PER_LEVEL, budget)
    for k, v in (opts or {}).items():
        it.set_option(k, v)
    cfg = O.Config(dim=dim, lower=lower, upper=upper, g=g, n_samples=n, trials=T, depth=depth, sigma_multiplier=m, seed=seed,
                   integrand=O.CONST, precision=precision, params=params, n_instances=n_instances, max_groups_per_level=budget)
    return it, cfg


def _compare(it, ores, n_samples, scale=1.0):
    """P2-P4 per component: sums within 1e-12*N*scale (only the FP64 summation order differs: the values are bit-identical),
    identical refined sets and cell identities, (mu, s, tau) and the results to rounding."""
    st = it.stats()
    assert st.overflow == 0
    n_cmp = 0
    for lev, ol in enumerate(ores.levels, start=1):
        gl = it.level_cells(lev)
        assert st.level[lev - 1].n_cells == ol.n_cells and st.level[lev - 1].n_refined == ol.n_refined
        np.testing.assert_array_equal(gl.instance, ol.instance)
        assert gl.path == ol.path
        assert gl.S.shape == ol.S.shape and gl.mu.shape == ol.mu.shape
        assert np.abs(gl.S - ol.S).max() <= 1e-12 * n_samples * scale
        sc = max(np.abs(ol.mu).max(), ol.s.max(), 1e-300)
        assert np.abs(gl.mu - ol.mu).max() <= 1e-11 * sc
        assert np.abs(gl.s - ol.s).max() <= 1e-9 * sc
        assert np.abs(gl.tau - ol.tau).max() <= 1e-9 * sc
        np.testing.assert_array_equal(gl.refined, ol.refined)
        n_cmp += ol.n_cells
    for lev in range(len(ores.levels) + 1, st.levels + 1):
        assert st.level[lev - 1].n_cells == 0
    v, s = it.result()
    assert v.shape == ores.value.shape
    assert np.all(np.abs(v - ores.value) <= 1e-11 * np.maximum(np.abs(ores.value), ores.std))
    assert np.all(np.abs(s - ores.std) <= 1e-9 * np.maximum(ores.std, 1e-300))
    return n_cmp


@pytest.mark.parametrize("precision", [O.F32, O.F64])
def test_poly4_whole_tree(precision):
    """Four polynomial components over [0,1]x[0,2]x[-1,1], depth 3, ragged N (not a multiple of the sample group)."""
    it, cfg = _make(3, [0, 0, -1], [1, 2, 1], 3, 1003, 5, 3, 1.0, 5, VS.POLY4, "poly4", 4, precision)
    it.run()
    ores = O.run_vec(cfg, 4, O.compile_user_fn(VS.POLY4, "poly4"), keep_cells=True)
    assert len(ores.levels) == 3 and ores.levels[1].n_refined > 0
    n = _compare(it, ores, 1003, scale=4.0)
    assert n == sum(l.n_cells for l in ores.levels)
    v, s = it.result()
    closed = np.array([2.0, 4.0 / 3.0, 12.0, 2.0])
    assert np.all(np.abs(v[0] - closed) <= 4 * s[0] + 1e-12)
    it.close()


def test_two_axes_union_rule_and_rerun():
    it, cfg = _make(2, [0, 0], [1, 2], 5, 3000, 5, 3, 1.0, 7, VS.TWO_AXES, "two_axes", 2, O.F32)
    it.run()
    ores = O.run_vec(cfg, 2, O.compile_user_fn(VS.TWO_AXES, "two_axes"), keep_cells=True)
    _compare(it, ores, 3000, scale=8.0)
    l1 = it.level_cells(1)
    flag = (l1.s > l1.tau).any(axis=1)
    only0, only1 = l1.s[:, 0] > l1.tau[:, 0], l1.s[:, 1] > l1.tau[:, 1]
    assert (only0 != only1).any() and only0.any() and only1.any()          # the union differs from either component's own set
    np.testing.assert_array_equal(l1.refined.astype(bool), flag)
    v0, s0 = it.result()
    it.run()                                                                # a second run of the same context: bit-identical
    v1, s1 = it.result()
    np.testing.assert_array_equal(v0, v1)
    np.testing.assert_array_equal(s0, s1)
    it.close()


def test_instances_with_budget_and_graph():
    p = np.array([[1.0], [2.5], [-0.5]])
    it, cfg = _make(2, [0, 0], [1, 2], 5, 2000, 4, 3, 0.5, 9, VS.SCALED_AXES, "scaled_axes", 2, O.F32, params=p, n_instances=3, budget=2)
    it.run()
    ores = O.run_vec(cfg, 2, O.compile_user_fn(VS.SCALED_AXES, "scaled_axes"), keep_cells=True)
    assert ores.levels[0].n_truncated > 0
    _compare(it, ores, 2000, scale=20.0)
    v0, s0 = it.result()
    assert v0.shape == (3, 2)
    it.set_option(B.OPT_USE_GRAPH, 1)
    it.run()
    v1, s1 = it.result()
    np.testing.assert_array_equal(v0, v1)
    np.testing.assert_array_equal(s0, s1)
    it.close()


def test_sibling_group_of_several_control_tiles():
    """k = 70^2 = 4900 cells per group: two 4096-cell control tiles, the three-launch threshold path, per component."""
    it, cfg = _make(2, [0, 0], [1, 2], 70, 64, 3, 2, 2.0, 3, VS.TWO_AXES, "two_axes", 2, O.F32, budget=3, cap=4 * 4900)
    it.run()
    ores = O.run_vec(cfg, 2, O.compile_user_fn(VS.TWO_AXES, "two_axes"), keep_cells=True)
    assert ores.levels[0].n_cells == 4900 and ores.levels[1].n_cells == 3 * 4900
    _compare(it, ores, 64, scale=8.0)
    it.close()


def test_one_component_through_the_vector_call_is_the_scalar_user_call():
    scalar_src = """
__device__ float axis0s(const float* x, int dim, const float* p, int np) { return x[0] * x[0]; }
__device__ double axis0s(const double* x, int dim, const double* p, int np) { return x[0] * x[0]; }
"""
    args = (2, [0, 0], [1, 2], 5, 3001, 5, 2, 1.0, 7)
    a = B.Integrator(*args)
    a.set_option(B.OPT_PRECISION, B.F32)
    a.set_integrand_source(scalar_src, "axis0s")
    a.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
    a.run()
    b = B.Integrator(*args)
    b.set_option(B.OPT_PRECISION, B.F32)
    b.set_integrand_source_vec(VS.AXIS0, "axis0", 1)
    b.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
    b.run()
    va, sa = a.result()
    vb, sb = b.result()
    assert vb.shape == (1, 1)
    assert abs(va[0] - vb[0, 0]) <= 1e-13 * abs(va[0]) and abs(sa[0] - sb[0, 0]) <= 1e-9 * sa[0]
    for lev in (1, 2):
        np.testing.assert_array_equal(a.level_cells(lev).refined, b.level_cells(lev).refined)
    a.close()
    b.close()


def test_moments8_6d_sampled_units_and_full_control():
    """Eight components over [0,1]^6, 4096 cells per group, budget 4: levels of 4096 and 16384 cells. Sampled (cell, trial)
    units against the oracle one by one (T2) and the whole control path re-derived in numpy from the dumped (mu, s) (T3)."""
    D, g, N, T, L, m, seed, C = 6, 4, 2001, 5, 2, 1.5, 21, 8
    p = np.array([[0.3]])
    it, cfg = _make(D, [0.0] * D, [1.0] * D, g, N, T, L, m, seed, VS.MOMENTS8, "moments8", C, O.F32, params=p, budget=4, cap=4 * 4096)
    it.run()
    v, s = it.result()
    st = it.stats()
    assert [st.level[l].n_cells for l in range(2)] == [4096, 4 * 4096]
    fns = O.compile_user_fn(VS.MOMENTS8, "moments8")
    rng = np.random.default_rng(5)
    k = g ** D
    acc_v, acc_q = np.zeros(C), np.zeros(C)
    for lev in (1, 2):
        gl = it.level_cells(lev)
        n = len(gl.refined)
        # T2: sampled units
        for cell in rng.integers(0, n, size=6):
            path = gl.path[cell]
            digits = []
            q = path
            for _ in range(lev):
                digits.append(q % k)
                q //= k
            P, coords = O.path_coords(D, g, digits[::-1])
            assert P == path
            t = int(rng.integers(0, T))
            S = O.vec_unit_sums(cfg, C, fns, 0, path, lev, coords, t)
            assert np.abs(gl.S[cell, t] - S).max() <= 1e-12 * N * 2.0
        # T3: (mu, s) from the dumped sums, tau, flags, budget, accepted sums
        V = (1.0 / g ** lev) ** D
        I = gl.S * V / N
        mu = I.mean(axis=1)
        sd = np.sqrt(((I - mu[:, None, :]) ** 2).mean(axis=1))
        np.testing.assert_allclose(gl.mu, mu, rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(gl.s, sd, rtol=1e-7, atol=1e-18)
        G = n // k
        sg = gl.s.reshape(G, k, C)
        mean = sg.mean(axis=1)
        tau = mean + m * np.sqrt(((sg - mean[:, None, :]) ** 2).mean(axis=1))
        np.testing.assert_allclose(gl.tau.reshape(G, k, C)[:, 0, :], tau, rtol=1e-11)
        flag = (gl.s > gl.tau).any(axis=1) & (lev < L)
        assert st.level[lev - 1].n_flagged == flag.sum()
        want = np.zeros(n, dtype=bool)
        want[np.nonzero(flag)[0][:4]] = True
        np.testing.assert_array_equal(gl.refined.astype(bool), want)
        acc_v += gl.mu[~want].sum(axis=0)
        acc_q += (gl.s[~want] ** 2).sum(axis=0)
    np.testing.assert_allclose(v[0], acc_v, rtol=1e-12)
    np.testing.assert_allclose(s[0], np.sqrt(acc_q), rtol=1e-10)
    # closed form of component 0: integral of 0.3 * sum x over the unit cube = 0.3 * 3
    assert abs(v[0, 0] - 0.9) <= 4 * s[0, 0]
    it.close()


@pytest.mark.parametrize("precision", [O.F32, O.F64])
def test_spread_from_samples_per_component(precision):
    """R13 + R15: sums of f_j^2 next to the sums of f_j, the spread of every component from its samples; whole tree against the oracle."""
    it, cfg = _make(3, [0, 0, -1], [1, 2, 1], 3, 1003, 4, 3, 0.5, 5, VS.POLY4, "poly4", 4, precision, budget=3,
                    opts={B.OPT_SPREAD: B.SPREAD_SAMPLES})
    cfg.spread = O.SPREAD_SAMPLES
    it.run()
    ores = O.run_vec(cfg, 4, O.compile_user_fn(VS.POLY4, "poly4"), keep_cells=True)
    assert len(ores.levels) == 3 and ores.levels[0].n_refined > 0
    _compare(it, ores, 1003, scale=4.0)
    for lev, ol in enumerate(ores.levels, start=1):
        Q = it.level_sumsq(lev, ol.n_cells)
        assert Q.shape == ol.Q.shape
        assert np.abs(Q - ol.Q).max() <= 1e-12 * 1003 * 16.0
    v, s = it.result()
    closed = np.array([2.0, 4.0 / 3.0, 12.0, 2.0])
    assert np.all(np.abs(v[0] - closed) <= 4.5 * s[0] + 1e-12)      # std is a 1-sigma error here
    assert s[0, 2] == 0.0                                            # the constant component
    it.close()


def test_error_states():
    it = B.Integrator(2, [0, 0], [1, 1], 3, 100, 3, 2, 1.0, 1)
    with pytest.raises(B.ZmcError) as e:
        it.set_integrand_source_vec(VS.TWO_AXES, "two_axes", 17)
    assert e.value.status == B.ERR_RANGE
    with pytest.raises(B.ZmcError) as e:
        it.set_integrand_source_vec(VS.TWO_AXES, "two_axes", 0)
    assert e.value.status == B.ERR_RANGE
    it.set_option(B.OPT_BUDGET_ORDER, B.BUDGET_LARGEST_SPREAD)
    with pytest.raises(B.ZmcError) as e:
        it.set_integrand_source_vec(VS.TWO_AXES, "two_axes", 2)
    assert e.value.status == B.ERR_STATE
    it.set_integrand_source_vec(VS.AXIS0, "axis0", 1)              # one component: a largest-spread budget is defined
    it.set_option(B.OPT_BUDGET_ORDER, B.BUDGET_PATH_ORDER)
    it.set_integrand_source_vec(VS.TWO_AXES, "two_axes", 2)
    with pytest.raises(B.ZmcError) as e:
        it.set_option(B.OPT_BUDGET_ORDER, B.BUDGET_LARGEST_SPREAD)
    assert e.value.status == B.ERR_STATE
    it.run()                                    # the context is still usable after the refusals
    v, s = it.result()
    assert v.shape == (1, 2) and np.all(np.isfinite(v)) and np.all(s > 0)
    # a compile error surfaces at the call, with the log
    with pytest.raises(B.ZmcError) as e:
        it.set_integrand_source_vec("__device__ void broken(", "broken", 2)
    assert e.value.status == B.ERR_COMPILE
    # back to a scalar built-in: results lose the component axis
    it.set_integrand(B.SIN_SUM)
    it.run()
    v, s = it.result()
    assert v.shape == (1,)
    it.close()


def test_bench_configuration_sampled_units_control_and_closed_forms():
    """The vector-valued bench workload at its full size (bench.py `vector_valued`: 6-D, 4096 cells, N = 1e5, T = 5, 8 components):
    sampled (cell, trial) units against the oracle, the control path re-derived in numpy, and all eight integrals against their
    closed forms -- the raw moments of a sum of six uniforms, exact rationals."""
    from fractions import Fraction
    from math import comb
    from paper_1902_07916_b200 import workloads as W
    w = W.vec_moments6d()
    C = 8
    it = B.Integrator(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.depth, w.sigma_multiplier, w.seed)
    it.set_option(B.OPT_PRECISION, B.F32)
    it.set_integrand_source_vec(W.VEC_MOMENTS_SRC, W.VEC_MOMENTS_FN, C, w.params, 1)
    it.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
    it.set_option(B.OPT_MAX_CELLS_PER_LEVEL, w.k)
    it.run()
    v, s = it.result()
    gl = it.level_cells(1)
    assert len(gl.refined) == 4096 and gl.refined.sum() == 0            # depth 1: nothing refined
    cfg = O.Config(dim=w.dim, lower=list(w.lower), upper=list(w.upper), g=w.g, n_samples=w.n_samples, trials=w.trials, depth=w.depth,
                   sigma_multiplier=w.sigma_multiplier, seed=w.seed, integrand=O.CONST, precision=O.F32, params=w.params)
    fns = O.compile_user_fn(W.VEC_MOMENTS_SRC, W.VEC_MOMENTS_FN)
    rng = np.random.default_rng(11)
    for cell in rng.integers(0, 4096, size=4):
        path, coords = O.path_coords(6, 4, [int(cell)])
        t = int(rng.integers(0, 5))
        S = O.vec_unit_sums(cfg, C, fns, 0, path, 1, coords, t)
        assert np.abs(gl.S[cell, t] - S).max() <= 1e-12 * w.n_samples * max(1.0, float(np.abs(S).max()) / w.n_samples)
    V = (1.0 / 4) ** 6
    I = gl.S * V / w.n_samples
    mu = I.mean(axis=1)
    np.testing.assert_allclose(gl.mu, mu, rtol=1e-12)
    np.testing.assert_allclose(v[0], gl.mu.sum(axis=0), rtol=1e-12)
    np.testing.assert_allclose(s[0], np.sqrt((gl.s ** 2).sum(axis=0)), rtol=1e-10)
    # E[(x1 + .. + x6)^j] for independent uniforms: M_n(j) = sum_m C(j, m) M_{n-1}(j - m) / (m + 1)
    M = [Fraction(1)] + [Fraction(0)] * C
    for _ in range(6):
        M = [sum(Fraction(comb(j, m)) * M[j - m] / (m + 1) for m in range(j + 1)) for j in range(C + 1)]
    closed = np.array([float(Fraction(3, 10) ** j * M[j]) for j in range(1, C + 1)])
    z = (v[0] - closed) / s[0]
    assert np.all(np.abs(z) < 4.0), z
    it.close()
