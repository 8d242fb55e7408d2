"""GPU parity for the two SURVEY 8(f).2 extensions (R13, R14), through the C ABI:
  ZMC_SPREAD_SAMPLES          the sampling kernel also sums f^2 (NVRTC-compiled SQ instance), cell spread from the samples;
  ZMC_BUDGET_LARGEST_SPREAD   device-side radix select of the B largest flagged spreads per instance.
Same rules as tests/test_gpu_parity.py: sums within 1e-12*N of the oracle's, identical refined sets, value within 1e-6."""
import math

import numpy as np
import pytest

import bench
import oracle as O
from paper_1902_07916_b200 import binding as B
from paper_1902_07916_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu

CASES = {
    "sin6_f32_ragged": W.config2().with_(n_samples=501, depth=2, max_groups_per_level=3),
    "gauss9_f32": W.config3().with_(n_samples=203, depth=3),
    "gauss4_batched": W.config4(n_instances=6).with_(n_samples=130, max_groups_per_level=2),
    "sin3_f64_chunks": W.Workload("s3c", 3, (0.0,) * 3, (10.0,) * 3, 2, 200003, 4, 2, 0.0, 10, W.SIN_SUM, W.F64),
    "sin5_f32": W.Workload("s5", 5, (0.0,) * 5, (4.0,) * 5, 3, 1022, 5, 2, 1.5, 7, W.SIN_SUM, W.F32, max_groups_per_level=2),
    "const3_f64": W.Workload("c3", 3, (0.0, 1.0, -1.0), (2.0, 3.0, 1.0), 3, 50, 4, 3, 1.5, 1, W.CONST, W.F64, params=np.array([[0.75]])),
}


def _both(w, spread, order):
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 18, spread=spread, budget_order=order)
    it.run()
    ores = O.run(H.oracle_config(w, spread=spread, budget_order=order), keep_cells=True)
    return it, ores


@pytest.mark.parametrize("name", sorted(CASES))
def test_sample_spread_whole_trees(name):
    w = CASES[name]
    it, ores = _both(w, B.SPREAD_SAMPLES, B.BUDGET_PATH_ORDER)
    H.compare_tree(it, ores, w)
    for lev, ol in enumerate(ores.levels, start=1):
        Q = it.level_sumsq(lev, ol.n_cells)
        assert np.abs(Q - ol.Q).max() <= 1e-12 * w.n_samples * max(1.0, float(np.abs(ol.Q).max()) / w.n_samples)
        if w.integrand == W.EXP_QUAD:
            assert np.all(np.abs(Q - ol.Q) <= 1e-12 * np.abs(ol.Q))
    if name == "const3_f64":
        assert np.all(it.level_cells(1).s == 0.0) and it.result()[1][0] == 0.0
    it.close()


@pytest.mark.parametrize("spread", [B.SPREAD_TRIALS, B.SPREAD_SAMPLES])
@pytest.mark.parametrize("name", ["gauss4_batched_m05", "sin6_small", "sin2_deep"])
def test_largest_spread_budget_whole_trees(name, spread):
    if name == "gauss4_batched_m05":
        w = W.config4(n_instances=5).with_(n_samples=150, depth=3, sigma_multiplier=0.5, max_groups_per_level=3)
    elif name == "sin6_small":
        w = W.config2().with_(n_samples=301, depth=3, max_groups_per_level=5)
    else:
        w = W.Workload("s2", 2, (0.0, 0.0), (7.0, 5.0), 5, 64, 5, 6, 0.3, 9, W.SIN_SUM, W.F64, max_groups_per_level=4)
    it, ores = _both(w, spread, B.BUDGET_LARGEST_SPREAD)
    H.compare_tree(it, ores, w)
    byp = O.run(H.oracle_config(w, spread=spread), keep_cells=True)
    assert any(not np.array_equal(a.refined, b.refined) for a, b in zip(ores.levels, byp.levels))   # the order matters here
    it.close()


def test_largest_spread_budget_with_many_instances():
    """With 64 instances or more (kSelectWideBelow in zmc_lib.cu) the radix select of R14 is ONE kernel with one block per instance
    (zmc_select_kernel) instead of the begin / histogram / pick launches over all tiles that every other R14 test takes (they have 1 to
    6 instances). 70 batched 4-D Gaussians, a binding budget of 2 cells per instance and level, three levels, against the oracle:
    pivot, quota and tile range of that kernel decide which cells are refined, so identical refined sets cover them."""
    w = W.config4(n_instances=70).with_(n_samples=40, depth=3, sigma_multiplier=0.5, max_groups_per_level=2)
    it, ores = _both(w, B.SPREAD_TRIALS, B.BUDGET_LARGEST_SPREAD)
    H.compare_tree(it, ores, w)
    st = it.stats()
    assert st.level[0].n_flagged > st.level[0].n_refined == 2 * w.n_instances       # every instance has at least 2 flagged cells, most far more: the budget binds
    assert st.level[1].n_flagged > st.level[1].n_refined == 2 * w.n_instances
    byp = O.run(H.oracle_config(w), keep_cells=True)
    assert any(not np.array_equal(a.refined, b.refined) for a, b in zip(ores.levels, byp.levels))   # and the order matters
    it.close()


def test_options_switch_kernels_and_layout():
    """Changing the spread after a run re-selects the kernel and re-lays the workspace; results match fresh contexts."""
    w = W.config1()
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 12)
    it.run()
    a = it.result()
    it.set_option(B.OPT_SPREAD, B.SPREAD_SAMPLES)
    it.run()
    b = it.result()
    ores = O.run(H.oracle_config(w, spread=O.SPREAD_SAMPLES))
    assert abs(b[0][0] - ores.value[0]) <= 1e-11 * abs(ores.value[0]) and abs(b[1][0] - ores.std[0]) <= 1e-9 * ores.std[0]
    it.set_option(B.OPT_SPREAD, B.SPREAD_TRIALS)
    it.run()
    c = it.result()
    assert a[0][0] == c[0][0] and a[1][0] == c[1][0]
    it.close()


def test_fullsize_sample_spread_and_largest_spread_budget():
    """BASELINE.json configs[1] at bench size with both extensions: sampled units (S and Q) against the oracle, every
    level's control re-derived in numpy (top-16 flagged spreads), and -- because std is now a 1-sigma error -- |z| < 4."""
    # m = 1.0: with the sample spread the per-cell s of f1 is nearly noise-free and bounded, and mean + 1.5 pstd lies above
    # its maximum (nothing would be flagged at all -- the chance refinement of SURVEY finding F1 is gone)
    w = bench.workloads()["cfg2_sin6d_depth3_B16"].with_(sigma_multiplier=1.0)
    cfg = H.oracle_config(w, spread=O.SPREAD_SAMPLES, budget_order=O.BUDGET_LARGEST_SPREAD)
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=bench.capacity_for(w), spread=B.SPREAD_SAMPLES,
                         budget_order=B.BUDGET_LARGEST_SPREAD)
    it.use_torch_workspace()
    it.run()
    v, sd = it.result()
    st = it.stats()
    rng = np.random.default_rng(5)
    k, T, N = w.k, w.trials, w.n_samples
    val = var = 0.0
    parents = None
    for level in range(1, w.depth + 1):
        gl = it.level_cells(level)
        n = len(gl.mu)
        Q = it.level_sumsq(level, n)
        if parents is not None:
            assert gl.path == [p * k + j for p in parents for j in range(k)]
        for c in rng.integers(0, n, size=6):
            t = int(rng.integers(0, T))
            digits = []
            p = gl.path[c]
            for _ in range(level):
                digits.append(p % k)
                p //= k
            path, coords = O.path_coords(w.dim, w.g, digits[::-1])
            S_o, Q_o = O.unit_sums(cfg, 0, path, level, coords, t)
            assert abs(gl.S[c, t] - S_o) <= 1e-12 * N and abs(Q[c, t] - Q_o) <= 1e-12 * N
        vol = math.prod((b - a) / w.g ** level for a, b in zip(w.lower, w.upper))
        M = float(T * N)
        Sc, Qc = gl.S.sum(axis=1), Q.sum(axis=1)
        d = Qc - Sc * Sc / M
        d[~(d > Qc * 2.0 ** -40)] = 0.0
        s = vol * np.sqrt(d / M / M)
        assert np.abs(gl.s - s).max() <= 1e-9 * s.max()
        tau_c, refined, lv, lvar = H.host_control(gl.mu, gl.s, k, level, w.depth, w.sigma_multiplier,
                                                  np.zeros(n, dtype=np.int64), budget=16, largest_spread=True)
        np.testing.assert_array_equal(gl.refined.astype(bool), refined)
        n_flagged = int(np.sum(gl.s > tau_c)) if level < w.depth else 0
        assert st.level[level - 1].n_refined == int(refined.sum()) == min(16, n_flagged)
        assert level == w.depth or n_flagged > 100          # the budget really selects
        val += lv[0]
        var += lvar[0]
        parents = [gl.path[i] for i in np.nonzero(refined)[0]]
    assert abs(v[0] - val) <= 1e-11 * max(abs(val), math.sqrt(var)) and abs(sd[0] - math.sqrt(var)) <= 1e-11 * math.sqrt(var)
    z = (v[0] - H.closed_sin_sum(w.lower, w.upper)) / sd[0]
    print("cfg2 with R13+R14: value %.6f +- %.4f, z = %.2f" % (v[0], sd[0], z))
    assert abs(z) < 4.0
    it.close()


def test_largest_spread_budget_with_exact_ties():
    """R14's tie rule (equal spreads are taken in ascending path order) cannot be reached with the built-in integrands: their
    spreads never coincide. A user integrand with two values -- stripes of width 1/37 in x0, N = 1, T = 2 -- makes every cell's
    spread exactly 0 or V/2, so dozens of flagged cells tie at the pivot. Checked against the brute-force selection in numpy
    (tests/helpers.py host_control) from the dumped (mu, s): pivot, quota and the path-order ranks among the ties."""
    src = r"""
    __device__ double stripes(const double* x, int dim, const double* p, int np) { return (double)(((int)(x[0] * 37.0)) & 1); }
    __device__ float stripes(const float* x, int dim, const float* p, int np) { return (float)(((int)(x[0] * 37.0f)) & 1); }
    """
    k, B_ = 64, 5
    it = B.Integrator(2, [0.0, 0.0], [1.0, 1.0], 8, 1, 2, 3, 0.0, 41)
    it.set_integrand_source(src, "stripes", None, 1)
    it.set_option(B.OPT_MAX_GROUPS_PER_LEVEL, B_)
    it.set_option(B.OPT_BUDGET_ORDER, B.BUDGET_LARGEST_SPREAD)
    it.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
    it.set_option(B.OPT_MAX_CELLS_PER_LEVEL, 1 << 12)
    it.run()
    v, s = it.result()
    parents = None
    tied_levels = 0
    for level in (1, 2, 3):
        gl = it.level_cells(level)
        n = len(gl.mu)
        assert n == (1 if level == 1 else B_) * k
        if parents is not None:
            assert gl.path == [p * k + j for p in parents for j in range(k)]
        V = (1.0 / 8 ** level) ** 2
        assert set(np.unique(gl.s)) <= {0.0, V / 2}                     # exact ties by construction
        tau_c, refined, lv, lvar = H.host_control(gl.mu, gl.s, k, level, 3, 0.0, np.zeros(n, dtype=np.int64), budget=B_,
                                                  largest_spread=True)
        flagged = gl.s > tau_c
        if level < 3:
            assert flagged.sum() > B_ and np.all(gl.s[flagged] == V / 2)
            tied_levels += 1
            assert list(np.nonzero(refined)[0]) == list(np.nonzero(flagged)[0][:B_])      # ties: first in path order
        np.testing.assert_array_equal(gl.refined.astype(bool), refined)
        parents = [gl.path[i] for i in np.nonzero(refined)[0]]
    assert tied_levels == 2
    it.close()


def test_largest_spread_budget_with_ties_below_larger_spreads():
    """As above with a three-valued integrand (0, 1, 3 in stripes): spreads are 0, V/2, V or 3V/2, so the pivot's ties sit below
    strictly larger spreads and only part of them fits the budget (quota < number of ties)."""
    src = r"""
    __device__ double steps(const double* x, int dim, const double* p, int np) { const int j = ((int)(x[0] * 53.0)) % 3; return j == 2 ? 3.0 : (double)j; }
    __device__ float steps(const float* x, int dim, const float* p, int np) { const int j = ((int)(x[0] * 53.0f)) % 3; return j == 2 ? 3.0f : (float)j; }
    """
    k, B_ = 64, 26      # this seed: 21 cells at 3V/2, then the ties at V
    it = B.Integrator(2, [0.0, 0.0], [1.0, 1.0], 8, 1, 2, 2, 0.0, 43)
    it.set_integrand_source(src, "steps", None, 1)
    it.set_option(B.OPT_MAX_GROUPS_PER_LEVEL, B_)
    it.set_option(B.OPT_BUDGET_ORDER, B.BUDGET_LARGEST_SPREAD)
    it.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
    it.set_option(B.OPT_MAX_CELLS_PER_LEVEL, 1 << 12)
    it.run()
    it.result()
    gl = it.level_cells(1)
    V = 1.0 / 64
    assert set(np.unique(gl.s)) <= {0.0, V / 2, V, 1.5 * V}
    tau_c, refined, _, _ = H.host_control(gl.mu, gl.s, k, 1, 2, 0.0, np.zeros(k, dtype=np.int64), budget=B_, largest_spread=True)
    flagged = gl.s > tau_c
    order = sorted(np.nonzero(flagged)[0], key=lambda i: (-gl.s[i], i))
    pivot = gl.s[order[B_ - 1]]
    n_greater = int(np.sum(gl.s[flagged] > pivot))
    n_ties = int(np.sum(gl.s[flagged] == pivot))
    assert 0 < n_greater < B_ and n_ties > B_ - n_greater, (n_greater, n_ties)        # the case the quota exists for
    np.testing.assert_array_equal(gl.refined.astype(bool), refined)
    assert it.level_cells(2).path == [int(p) * k + j for p in np.nonzero(refined)[0] for j in range(k)]
    it.close()
