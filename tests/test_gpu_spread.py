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
