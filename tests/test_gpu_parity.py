"""GPU parity tests proper: the CUDA path (through the C ABI of include/zmc.h, via the ctypes binding)
against the oracle, element by element on the same seeded inputs (parity rules P1-P4, DESIGN.md
section 5). Every test here needs a B200 and is marked gpu.

Tolerances (derived from the arithmetic):
  * Philox words, FP32 points and FP32 integrand values: bit-exact (integer work / the same IEEE
    operation sequence on both sides, R8).
  * FP64 points: bit-exact (same +,* sequence); FP64 sin/exp values: <= 4 ulp (libm vs CUDA libdevice).
  * per-(cell,trial) sums: BASELINE.json asks 1e-6 relative; only the FP64 summation order differs,
    so exact mode is held to 1e-12 * N (N terms each <= 1 in magnitude, error <= N * 2^-53 * log-ish).
  * refined-cell sets: identical. Final integral: 1e-6 relative (BASELINE.json), in fact ~1e-13.
"""
import numpy as np
import pytest

import oracle as O
from paper_1902_07916_b200 import binding as B
from paper_1902_07916_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _run_both(w, math=B.MATH_EXACT, max_cells=1 << 18):
    it = B.from_workload(w, math=math, keep_level_stats=True, max_cells_per_level=max_cells)
    it.run()
    ores = O.run(H.oracle_config(w), keep_cells=True)
    return it, ores


# ------------------------------------------------------------------ P1: generator, map, integrand
def test_philox_words_bit_exact():
    w = W.config4(n_instances=5)
    with B.from_workload(w) as it:
        cases = [(0, 0, 1, 0, 0, 4096), (3, 12345, 2, 4, 17, 1001), (4, (1 << 79) + (1 << 64) + 99, 15, 254, 3, 515),
                 (1, (1 << 64) - 1, 7, 1, (1 << 33) + 2, 64), (2, 0x0123456789ABCDEF, 3, 2, 4 * ((1 << 32) - 8), 32)]
        for inst, path, level, trial, first, n in cases:
            g = it.debug_words(inst, path, level, trial, first, n)
            o = O.unit_words(w.seed, inst, path, level, trial, first, n)
            np.testing.assert_array_equal(g, o)


@pytest.mark.parametrize("name", ["sin6_f32", "gauss9_f32", "gauss4_f32_batched", "linear5_f32", "const2_f32",
                                  "sin3_f64", "gauss9_f64", "linear7_f64"])
def test_points_and_values(name):
    rng = np.random.default_rng(11)
    if name == "sin6_f32":
        w = W.config2()
    elif name == "gauss9_f32":
        w = W.config3()
    elif name == "gauss4_f32_batched":
        w = W.config4(n_instances=3)
    elif name == "linear5_f32":
        w = W.Workload("lin5", 5, (-1.0, 0.0, 2.0, -3.0, 0.5), (1.0, 0.25, 7.0, -1.0, 0.75), 3, 100, 3, 3, 1.5, 9,
                       W.LINEAR, W.F32, params=rng.normal(size=(1, 6)))
    elif name == "const2_f32":
        w = W.Workload("c2", 2, (0.0, 0.0), (1.0, 2.0), 2, 10, 2, 1, 1.5, 9, W.CONST, W.F32, params=np.array([[0.3]]))
    elif name == "sin3_f64":
        w = W.config1()
    elif name == "gauss9_f64":
        w = W.config3().with_(precision=W.F64)
    else:
        w = W.Workload("lin7", 7, (0.0,) * 7, (1.0, 2.0, 3.0, 4.0, 5.0, 6.0, 7.0), 2, 100, 3, 3, 1.5, 9,
                       W.LINEAR, W.F64, params=rng.normal(size=(1, 8)))
    cfg = H.oracle_config(w)
    n = 999
    with B.from_workload(w) as it:
        for level in (1, w.depth):
            digits = [int(rng.integers(0, w.k)) for _ in range(level)]
            if name.startswith("gauss9"):
                digits = [(w.k - 1) // 2] * level      # the centre cell, where the values are not all zero
            path, coords = O.path_coords(w.dim, w.g, digits)
            inst = w.n_instances - 1
            trial = w.trials - 1
            xg, fg = it.debug_points(inst, path, level, coords, trial, n)
            xo, fo = O.unit_points(cfg, inst, path, level, coords, trial, n)
            np.testing.assert_array_equal(xg, xo)
            if w.precision == W.F32 or w.integrand in (W.CONST, W.LINEAR):
                np.testing.assert_array_equal(fg, fo)
            else:
                assert np.all(np.abs(fg - fo) <= 4 * np.spacing(np.abs(fo)))
            if name.startswith("gauss9") and level > 1:
                assert np.count_nonzero(fo) > n // 2


def test_fast_mode_values_close():
    """MUFU mode (R8): not bit-comparable; |sin| error <= 2^-21.4 on [-pi,pi] scaled by the range
    reduction inside __sinf (abs error <= 4e-6 measured for |a| <= 60, bound 1e-5); exp relative error <= 1e-6."""
    for w, tol in ((W.config2(), 1e-5), (W.config4(n_instances=2), 2e-6)):
        cfg = H.oracle_config(w)
        path, coords = O.path_coords(w.dim, w.g, [w.k // 3])
        with B.from_workload(w, math=B.MATH_FAST) as it:
            xg, fg = it.debug_points(0, path, 1, coords, 0, 2000)
        xo, fo = O.unit_points(cfg, 0, path, 1, coords, 0, 2000)
        np.testing.assert_array_equal(xg, xo)
        if w.integrand == W.SIN_SUM:
            assert np.abs(fg - fo).max() <= tol
        else:
            # e*log2(e) is rounded once in FP32 before MUFU.EX2: relative error ~ |e| * 2^-24 on top of EX2's 2^-22
            assert np.all(np.abs(fg - fo) <= (tol + 1.5e-7 * np.abs(np.log(fo))) * np.abs(fo))


# ------------------------------------------------------------------ P2-P4: whole trees, small enough for the oracle
def test_config1_whole_tree():
    """BASELINE.json configs[0] end to end, all 64 + 5*64 cells, 1920 (cell,trial) sums."""
    w = W.config1()
    it, ores = _run_both(w)
    n = H.compare_tree(it, ores, w)
    assert n == 64 + 5 * 64
    assert sorted(np.nonzero(it.level_cells(1).refined)[0].tolist()) == [1, 24, 26, 34, 41]   # golden/config1_worked.txt
    v, s = it.result()
    closed = H.closed_sin_sum(w.lower, w.upper)
    assert abs(v[0] - closed) <= 4 * s[0]
    it.close()


SMALL = {
    # 6-D sin, FP32 exact: several tiles of cells, ragged sample count (N odd: last group half full), budget
    "sin6_f32_ragged": W.config2().with_(n_samples=501, depth=2, max_groups_per_level=3),
    # 9-D Gaussian, FP32 extended range: one refined cell per level, depth 3
    "gauss9_f32": W.config3().with_(n_samples=203, depth=3),
    # batched 4-D Gaussians: 6 instances, own keys / thresholds / budgets
    "gauss4_batched": W.config4(n_instances=6).with_(n_samples=130, max_groups_per_level=2),
    # FP64 Gaussian, D=2, deep tree without budget
    "gauss2_f64_deep": W.Workload("g2", 2, (-1.0, -2.0), (1.5, 1.0), 3, 97, 4, 5, 0.5, 21, W.EXP_QUAD, W.F64,
                                  params=np.array([[2.0, 40.0, 0.1, -0.3]])),
    # D=1 and D=4 (a whole Philox call per sample), D=5 (4 samples per 5 calls), D=7, D=12
    "sin1_f32": W.Workload("s1", 1, (0.0,), (3.0,), 7, 1001, 6, 3, 1.0, 5, W.SIN_SUM, W.F32),
    "sin4_f64": W.Workload("s4", 4, (0.0,) * 4, (2.0,) * 4, 3, 63, 3, 2, 1.0, 6, W.SIN_SUM, W.F64),
    "sin5_f32": W.Workload("s5", 5, (0.0,) * 5, (4.0,) * 5, 3, 1022, 5, 2, 1.5, 7, W.SIN_SUM, W.F32, max_groups_per_level=2),
    "sin7_f32": W.Workload("s7", 7, (0.0,) * 7, (4.0,) * 7, 2, 333, 5, 3, 1.0, 8, W.SIN_SUM, W.F32, max_groups_per_level=5),
    "lin12_f32": W.Workload("l12", 12, (0.0,) * 12, (1.0,) * 12, 2, 17, 3, 2, 1.0, 9, W.LINEAR, W.F32,
                            params=np.linspace(-1, 1, 13)[None, :], max_groups_per_level=1),
    # long units: N large enough that a unit is split into sample chunks (few cells, many samples)
    "sin3_f64_chunks": W.Workload("s3c", 3, (0.0,) * 3, (10.0,) * 3, 2, 200003, 4, 2, 0.0, 10, W.SIN_SUM, W.F64),
    "sin6_f32_chunks": W.Workload("s6c", 6, (0.0,) * 6, (10.0,) * 6, 1, 1000001, 3, 1, 1.5, 12, W.SIN_SUM, W.F32),
}


@pytest.mark.parametrize("name", sorted(SMALL))
def test_small_whole_trees(name):
    w = SMALL[name]
    it, ores = _run_both(w)
    H.compare_tree(it, ores, w)
    if w.integrand == W.EXP_QUAD:   # sums span hundreds of decades: also compare each sum relative to itself (f >= 0)
        for lev, ol in enumerate(ores.levels, start=1):
            gl = it.level_cells(lev)
            assert np.all(np.abs(gl.S - ol.S) <= 1e-12 * np.abs(ol.S))
    it.close()


def test_path_beyond_64_bits():
    """D=11, g=2, depth 7: paths reach 77 bits (R2: 80-bit path in the Philox counter)."""
    w = W.Workload("deep11", 11, (0.0,) * 11, (1.0,) * 11, 2, 8, 3, 7, 0.0, 13, W.LINEAR, W.F32,
                   params=np.linspace(0.5, 2, 12)[None, :], max_groups_per_level=1)
    it, ores = _run_both(w)
    H.compare_tree(it, ores, w)
    assert len(ores.levels) == 7 and max(ores.levels[6].path) >= 1 << 64
    it.close()


def test_fast_mode_whole_tree_within_bj_tolerance():
    """P2 in fast mode: sums within 1e-6 relative to sum|f| <= N; P3/P4 as far as fast mode allows:
    a refined-set difference is tolerated only for cells within the propagated deviation of tau."""
    w = W.config2().with_(n_samples=2000, depth=2, max_groups_per_level=2)
    it = B.from_workload(w, math=B.MATH_FAST, keep_level_stats=True, max_cells_per_level=1 << 16)
    it.run()
    ores = O.run(H.oracle_config(w), keep_cells=True)
    g1, o1 = it.level_cells(1), ores.levels[0]
    assert np.abs(g1.S - o1.S).max() <= 1e-6 * w.n_samples
    diff = np.nonzero(g1.refined != o1.refined)[0]
    V = (10.0 / 4) ** 6
    delta = np.abs(g1.S - o1.S).max(axis=1) * V / w.n_samples + np.abs(g1.tau - o1.tau)
    for c in diff:
        assert abs(o1.s[c] - o1.tau[c]) <= 4 * delta[c] + 1e-6 * o1.tau[c]
    if len(diff) == 0:
        # every unit sum is within 1e-6 * sum|f| <= 1e-6 * N, so the integral is within 1e-6 * Vol * max|f|
        # (the signed value suffers cancellation: -122 on a domain of volume 1e6); observed ~1e-9 * Vol
        v, s = it.result()
        assert abs(v[0] - ores.value[0]) <= 1e-6 * 10.0 ** 6
        assert abs(v[0] - ores.value[0]) <= 1e-4 * ores.std[0]
    it.close()


# ------------------------------------------------------------------ degenerate cases (R7)
def test_degenerate_cases():
    # CONST: every s is 0 -> tau = 0 -> nothing flagged (0 > 0 is false); value = c * Vol; std = 0
    w = W.Workload("c3", 3, (0.0, 1.0, -1.0), (2.0, 3.0, 1.0), 3, 50, 4, 3, 1.5, 1, W.CONST, W.F64, params=np.array([[0.75]]))
    it, ores = _run_both(w)
    H.compare_tree(it, ores, w)
    v, s = it.result()
    assert abs(v[0] - 0.75 * 8.0) < 1e-12 and s[0] == 0.0
    assert it.stats().level[1].n_cells == 0
    it.close()
    # g = 1 (k = 1): one cell per group, s = tau, never flagged; T = 1: every s = 0; N = 1; depth 1
    for kw in (dict(g=1, depth=3), dict(trials=1, depth=3), dict(n_samples=1, depth=2), dict(depth=1),
               dict(n_samples=3, depth=2)):
        w = W.config1().with_(**kw)
        it, ores = _run_both(w)
        H.compare_tree(it, ores, w)
        it.close()


def test_counter_field_limits():
    """R3 limits: trial index up to 254 (T = 255, 8 bits) and level 15 (4 bits) reach the Philox counter intact."""
    w = W.Workload("t255", 2, (0.0, 0.0), (1.0, 2.0), 2, 7, 255, 2, 1.0, 77, W.SIN_SUM, W.F32)
    it, ores = _run_both(w)
    H.compare_tree(it, ores, w)
    it.close()
    w = W.Workload("l15", 1, (0.0,), (3.0,), 2, 9, 3, 15, 0.0, 78, W.SIN_SUM, W.F64)
    it, ores = _run_both(w)
    H.compare_tree(it, ores, w)
    assert len(ores.levels) == 15 and it.stats().level[14].n_cells == 2
    it.close()


def test_nan_is_accepted_and_counted():
    """R7: NaN s compares false -> accepted; result NaN; counted in zmc_stats.nonfinite."""
    w = W.Workload("nan", 2, (0.0, 0.0), (1.0, 1.0), 2, 16, 3, 2, 1.0, 1, W.CONST, W.F64, params=np.array([[np.nan]]))
    with B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 12) as it:
        it.run()
        v, s = it.result()
        assert np.isnan(v[0])
        st = it.stats()
        assert st.nonfinite == 4 and st.level[0].n_refined == 0


def test_capacity_overflow_is_reported():
    w = W.config1().with_(sigma_multiplier=-10.0, depth=3)     # tau below every s: all 64 cells flagged
    with B.from_workload(w, max_cells_per_level=64 * 8) as it:  # room for 8 parents only
        it.run()
        with pytest.raises(B.ZmcError) as e:
            it.result()
        assert e.value.status == B.ERR_CAPACITY
        assert it.stats().overflow == 1


def test_rerun_is_bit_identical_and_workspace_from_torch():
    import torch
    w = W.config1()
    with B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 12) as it:
        it.use_torch_workspace()
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            it.run()
            a = it.result()
            c1 = it.level_cells(2)
            it.run()
            b = it.result()
            c2 = it.level_cells(2)
        assert a[0][0] == b[0][0] and a[1][0] == b[1][0]
        np.testing.assert_array_equal(c1.S, c2.S)
        np.testing.assert_array_equal(c1.mu, c2.mu)


# ------------------------------------------------------------------ user integrand (NVRTC, sm_100a)
USER_SRC = r"""
__device__ double my_f(const double* x, int dim, const double* p, int np) {
    double a = 0.0;
    for (int d = 0; d < dim; ++d) a += x[d];
    return p[0] * sin(a);
}
__device__ float my_f(const float* x, int dim, const float* p, int np) {
    float a = 0.0f;
    for (int d = 0; d < dim; ++d) a += x[d];
    return p[0] * sinf(a);
}
"""


def test_user_integrand_jit():
    w = W.config1()
    closed = 2.0 * H.closed_sin_sum(w.lower, w.upper)
    for prec in (B.F64, B.F32):
        it = B.Integrator(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.depth, w.sigma_multiplier, w.seed)
        it.set_option(B.OPT_PRECISION, prec)
        it.set_integrand_source(USER_SRC, "my_f", np.array([[2.0]]), 1)
        it.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
        it.set_option(B.OPT_MAX_CELLS_PER_LEVEL, 1 << 12)
        it.run()
        v, s = it.result()
        assert abs(v[0] - closed) <= 4 * s[0]
        if prec == B.F64:   # same points, same sums as the built-in up to the factor 2 and sin's last ulp
            ores = O.run(H.oracle_config(w), keep_cells=True)
            g1 = it.level_cells(1)
            assert np.abs(g1.S - 2.0 * ores.levels[0].S).max() <= 1e-10 * w.n_samples
            np.testing.assert_array_equal(g1.refined, ores.levels[0].refined)
        it.close()
    it = B.Integrator(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.depth, w.sigma_multiplier, w.seed)
    with pytest.raises(B.ZmcError) as e:
        it.set_integrand_source("__device__ double broken(const double* x, int d, const double* p, int n) { return y; }",
                                "broken", None, 1)
    assert e.value.status == B.ERR_COMPILE and "error" in str(e.value)
    it.close()


def test_dimension_above_aot_range_is_jitted():
    """13 <= D <= 16 has no pre-compiled kernel: the built-in is JIT-compiled from the same device source."""
    w = W.Workload("l13", 13, (0.0,) * 13, (1.0,) * 13, 1, 64, 3, 1, 1.0, 3, W.LINEAR, W.F32,
                   params=np.linspace(-1, 1, 14)[None, :])
    it, ores = _run_both(w)
    H.compare_tree(it, ores, w)
    it.close()


def test_jit_cache_skips_nvrtc_for_the_same_source():
    """A second context with the same user source reuses the compiled cubin (process-wide cache keyed by the program text)."""
    import time
    w = W.config1()
    src = USER_SRC.replace("my_f", "my_cached_f")
    times, origins = [], []
    for _ in range(2):
        it = B.Integrator(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.depth, w.sigma_multiplier, w.seed)
        t0 = time.perf_counter()
        it.set_integrand_source(src, "my_cached_f", np.array([[2.0]]), 1)
        times.append(time.perf_counter() - t0)
        it.run()
        v, s = it.result()
        assert abs(v[0] - 2.0 * H.closed_sin_sum(w.lower, w.upper)) <= 4 * s[0]
        origins.append(it.stats().kernel_origin)
        it.close()
    assert origins == [1, 2], (origins, times)      # compiled, then served from the process-wide cache


def test_graph_mode_is_bit_identical():
    """ZMC_OPT_USE_GRAPH: the whole run replayed as one CUDA graph gives the same bits as the kernel-by-kernel run,
    on the default stream and on a side stream, run after run; an option change re-captures."""
    import torch
    for w in (W.config1(), W.config2().with_(n_samples=333, depth=3, max_groups_per_level=2)):
        ref = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 15)
        ref.run()
        rv, rs = ref.result()
        it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 15, use_graph=True, single_launch=0)    # these small trees would take the single launch
        for rep in range(3):
            it.run()
            v, s = it.result()
            assert v[0] == rv[0] and s[0] == rs[0]
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            it.run()
            v, s = it.result()
        assert v[0] == rv[0] and s[0] == rs[0]
        for lev in range(1, w.depth + 1):
            a, b = it.level_cells(lev), ref.level_cells(lev)
            np.testing.assert_array_equal(a.S, b.S)
            np.testing.assert_array_equal(a.refined, b.refined)
        st = it.stats()
        assert st.total_ms > 0 and st.level[0].sample_ms == 0.0
        it.set_option(B.OPT_MAX_GROUPS_PER_LEVEL, 1)          # drops the graph; the next run captures the new parameters
        it.run()
        v2, _ = it.result()
        w1 = w.with_(max_groups_per_level=1)
        chk = B.from_workload(w1, max_cells_per_level=1 << 15)
        chk.run()
        assert v2[0] == chk.result()[0][0]
        for x in (ref, it, chk):
            x.close()


def test_user_integrand_parameter_sweep():
    """one user function, many parameter sets (n_instances > 1): each instance has its own key, thresholds
    and result. f_b(x) = exp(-a_b |x - c_b|^2) written as user source must reproduce the built-in EXP_QUAD instance by
    instance in FP64 (same points; exp from the same libdevice), and match the closed forms."""
    w = W.config4(n_instances=5).with_(n_samples=300, precision=W.F64, max_groups_per_level=2)
    src = r"""
    __device__ double sweep_f(const double* x, int dim, const double* p, int np) {
        double q = 0.0;
        for (int d = 0; d < dim; ++d) { const double y = x[d] - p[2 + d]; q += y * y; }
        return p[0] * exp(-(p[1] * q));
    }
    __device__ float sweep_f(const float* x, int dim, const float* p, int np) { return 0.0f; }
    """
    ref = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 16)
    ref.run()
    rv, rs = ref.result()
    it = B.Integrator(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.depth, w.sigma_multiplier, w.seed)
    it.set_option(B.OPT_PRECISION, B.F64)
    it.set_integrand_source(src, "sweep_f", w.params, w.n_instances)
    it.set_option(B.OPT_MAX_GROUPS_PER_LEVEL, 2)
    it.set_option(B.OPT_KEEP_LEVEL_STATS, 1)
    it.set_option(B.OPT_MAX_CELLS_PER_LEVEL, 1 << 16)
    it.run()
    v, s = it.result()
    # the built-in applies the prefactor p[0] = 1 per trial and contracts nothing; the user code may be contracted by NVRTC? no:
    # --fmad=false. q is summed in the same order, so the sums agree to the last few ulps of exp.
    assert np.all(np.abs(v - rv) <= 1e-12 * np.abs(rv)) and np.all(np.abs(s - rs) <= 1e-9 * rs)
    np.testing.assert_array_equal(it.level_cells(1).refined, ref.level_cells(1).refined)
    for b in range(w.n_instances):
        assert abs(v[b] - H.closed_exp_quad(w.params[b], w.lower, w.upper)) <= 4 * s[b]
    it.close()
    ref.close()


def test_maximum_sample_count():
    """The largest N the counter layout allows (R3: N*D/4 < 2^32 - 4096): D = 1, one cell, N = 2^34 - 2^15 samples per trial,
    cut into 65536 chunks. Too many for the oracle; the words at the top of the index range are compared bit for bit, and the
    integral of sin over [0, 3] must come out within 4 sigma at a spread of ~1e-5 (a wrapped or skipped index range would
    show as a wrong sample count in the estimate's scale)."""
    N = (1 << 34) - (1 << 15)
    w = W.Workload("nmax", 1, (0.0,), (3.0,), 1, N, 3, 1, 1.0, 31, W.SIN_SUM, W.F32)
    with B.from_workload(w, keep_level_stats=True, max_cells_per_level=16) as it:
        g = it.debug_words(0, 0, 1, 2, N - 64, 64)
        o = O.unit_words(w.seed, 0, 0, 1, 2, N - 64, 64)
        np.testing.assert_array_equal(g, o)
        it.run()
        v, s = it.result()
        S = it.level_cells(1).S[0]
        closed = 1.0 - np.cos(3.0)
        assert abs(v[0] - closed) <= 4 * s[0] + 1e-7 and s[0] < 2e-5       # 1e-7: the FP32 lattice and zsin's own error
        # each trial's mean of f is 3 * S / N; three independent estimates agree to a few 1e-5
        assert np.all(np.abs(3.0 * S / N - closed) < 6e-5)
    with pytest.raises(B.ZmcError) as e:
        B.Integrator(1, [0.0], [3.0], 1, 1 << 34, 3, 1, 1.0, 31)
    assert e.value.status == B.ERR_RANGE


def test_many_instances():
    """3000 independent instances with their own keys, parameters, thresholds and budgets (R11): per-instance scans,
    first/last group bookkeeping and results at a count well above one CTA's width."""
    rng = np.random.default_rng(3)
    n = 3000
    p = np.empty((n, 4))
    p[:, 0] = 1.0
    p[:, 1] = (10.0 ** rng.uniform(0, 2, n)).astype(np.float32)
    p[:, 2:] = (0.2 + 0.6 * rng.random((n, 2))).astype(np.float32)
    w = W.Workload("many", 2, (0.0, 0.0), (1.0, 1.0), 3, 48, 3, 3, 0.7, 17, W.EXP_QUAD, W.F32, params=p, n_instances=n,
                   max_groups_per_level=2)
    it, ores = _run_both(w, max_cells=n * 9 * 4)
    H.compare_tree(it, ores, w)
    assert ores.levels[1].n_cells > n * 9 and len(ores.levels) == 3
    it.close()


def test_impossible_size_is_an_error_not_a_crash():
    """k = 16^10 = 2^40 cells at level 1 passes the range checks but cannot be allocated: zmc_run reports it."""
    w = W.Workload("huge", 10, (0.0,) * 10, (1.0,) * 10, 16, 4, 2, 1, 1.0, 1, W.SIN_SUM, W.F32)
    it = B.from_workload(w)
    with pytest.raises(B.ZmcError) as e:
        it.run()
    assert e.value.status in (B.ERR_CUDA, B.ERR_CAPACITY, B.ERR_RANGE)
    it.close()
    # and the library still works afterwards
    w1 = W.config1()
    it = B.from_workload(w1)
    it.run()
    assert abs(it.result()[0][0] - (-4.553120732569151)) < 1e-9
    it.close()


def test_capacity_boundary_and_grid_independence():
    """Exactly enough room is enough (5 refined cells of config 1 -> 5 parents); one fewer is an overflow. The result does
    not depend on the size of the persistent grid (1 CTA, 7 CTAs, the default), bit for bit."""
    w = W.config1()
    ref = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 12)
    ref.run()
    rv, rs = ref.result()
    rS = ref.level_cells(2).S
    for cap, ok in ((5 * 64, True), (4 * 64, False)):
        it = B.from_workload(w, max_cells_per_level=cap)
        it.run()
        if ok:
            v, s = it.result()
            assert v[0] == rv[0] and s[0] == rs[0]
        else:
            with pytest.raises(B.ZmcError) as e:
                it.result()
            assert e.value.status == B.ERR_CAPACITY
        it.close()
    for grid in (1, 7):
        it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 12)
        it.set_option(B.OPT_GRID_BLOCKS, grid)
        it.run()
        v, s = it.result()
        assert v[0] == rv[0] and s[0] == rs[0] and it.stats().grid_blocks == grid
        np.testing.assert_array_equal(it.level_cells(2).S, rS)
        it.close()
    # a different chunking changes the summation order only
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 12)
    it.set_option(B.OPT_TARGET_ITEMS, 320)
    it.run()
    v, s = it.result()
    assert abs(v[0] - rv[0]) <= 1e-12 * abs(rv[0]) and np.abs(it.level_cells(2).S - rS).max() <= 1e-12 * w.n_samples
    it.close()
    ref.close()


def test_api_state_errors_and_context_reuse():
    w = W.config1()
    it = B.Integrator(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.depth, w.sigma_multiplier, w.seed)
    with pytest.raises(B.ZmcError) as e:
        it.run()
    assert e.value.status == B.ERR_NO_INTEGRAND
    with pytest.raises(B.ZmcError) as e:
        it.workspace_bytes()
    assert e.value.status == B.ERR_NO_INTEGRAND
    it.set_integrand(B.SIN_SUM)
    with pytest.raises(B.ZmcError) as e:
        it.result()
    assert e.value.status == B.ERR_NOT_RUN
    with pytest.raises(B.ZmcError) as e:
        it.set_integrand(B.EXP_QUAD, np.array([[1.0, 2.0]]), 1)        # too few parameters for D = 3
    assert e.value.status == B.ERR_ARG
    with pytest.raises(B.ZmcError) as e:
        it.set_option(99, 1)
    assert e.value.status == B.ERR_ARG
    with pytest.raises(B.ZmcError) as e:
        it.set_workspace(256, 1 << 20) if False else it.set_workspace(257, 1 << 20)     # not 256-byte aligned
    assert e.value.status == B.ERR_ARG
    it.run()
    a = it.result()
    with pytest.raises(B.ZmcError) as e:
        it.level_cells(1)                                              # level stats were not kept
    assert e.value.status == B.ERR_STATE
    # the same context, another integrand and instance count
    p = W.batched_params(4, 3, 9)
    it.set_integrand(B.EXP_QUAD, p, 4)
    it.set_option(B.OPT_PRECISION, B.F32)
    it.run()
    v, s = it.result()
    for b in range(4):
        assert abs(v[b] - H.closed_exp_quad(p[b], w.lower, w.upper)) <= 4 * s[b]
    # and back: bit-identical to the first run
    it.set_integrand(B.SIN_SUM)
    it.set_option(B.OPT_PRECISION, B.F64)
    it.run()
    b2 = it.result()
    assert a[0][0] == b2[0][0] and a[1][0] == b2[1][0]
    it.close()
    # a workspace that is too small is refused at run time
    import torch
    it = B.from_workload(w)
    buf = torch.empty(4096, dtype=torch.uint8, device="cuda")
    it.set_workspace((buf.data_ptr() + 255) & ~255, 1024)
    with pytest.raises(B.ZmcError) as e:
        it.run()
    assert e.value.status == B.ERR_ARG
    it.close()


def test_wide_groups_and_maximum_dimension():
    """k = 60000 cells per sibling group in one dimension (234 compaction tiles per group, integer coordinates up to 3.6e9 at
    level 2), and D = 16 = ZMC_MAX_DIM with 65536 cells (NVRTC instance, 4 Philox calls per sample)."""
    w = W.Workload("wide", 1, (-2.0,), (5.0,), 60000, 8, 3, 2, 1.0, 23, W.SIN_SUM, W.F64, max_groups_per_level=3)
    it, ores = _run_both(w, max_cells=4 * 60000)
    H.compare_tree(it, ores, w)
    assert ores.levels[1].n_cells == 3 * 60000
    it.close()
    for prec, integrand, params in ((W.F32, W.LINEAR, np.linspace(-1.0, 1.0, 17)[None, :]), (W.F64, W.SIN_SUM, None)):
        w = W.Workload("d16", 16, (0.0,) * 16, (1.0,) * 16, 2, 9, 3, 1, 1.0, 29, integrand, prec, params=params)
        it, ores = _run_both(w)
        H.compare_tree(it, ores, w)
        it.close()


def test_two_contexts_on_two_streams():
    """Distinct contexts are independent: two tree searches enqueued on two streams at the same time, several times over,
    give the results each gives alone."""
    import torch
    wa = W.config2().with_(n_samples=3001, depth=2, max_groups_per_level=2)
    wb = W.config3().with_(n_samples=1500, depth=3)
    alone = []
    for w in (wa, wb):
        with B.from_workload(w, max_cells_per_level=1 << 17) as it:
            it.run()
            alone.append(it.result())
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ia = B.from_workload(wa, max_cells_per_level=1 << 17)
    ib = B.from_workload(wb, max_cells_per_level=1 << 17)
    for _ in range(3):
        ia.run(sa.cuda_stream)
        ib.run(sb.cuda_stream)
        ra, rb = ia.result(), ib.result()
        assert ra[0][0] == alone[0][0][0] and ra[1][0] == alone[0][1][0]
        assert rb[0][0] == alone[1][0][0] and rb[1][0] == alone[1][1][0]
    ia.close()
    ib.close()


def test_disk_cache_of_compiled_integrands(tmp_path):
    """ZMC_CACHE_DIR: a second *process* with the same user source loads the cubin from disk instead of calling NVRTC;
    a corrupted file is ignored (and replaced). The directory is this test's own, so nothing depends on earlier runs."""
    import os
    import subprocess
    import sys
    script = r'''
import sys, time
sys.path.insert(0, %r)
import numpy as np
from paper_1902_07916_b200 import binding as B
SRC = """
__device__ double cached_g(const double* x, int dim, const double* p, int np) { return p[0] * x[0] * x[1]; }
__device__ float cached_g(const float* x, int dim, const float* p, int np) { return p[0] * x[0] * x[1]; }
"""
it = B.Integrator(2, [0.0, 0.0], [1.0, 2.0], 3, 500, 4, 2, 1.0, 3)
t0 = time.perf_counter()
it.set_integrand_source(SRC, "cached_g", np.array([[3.0]]), 1)
dt = time.perf_counter() - t0
it.run()
v, s = it.result()
assert abs(v[0] - 3.0) <= 4 * s[0], (v, s)          # integral of 3xy over [0,1]x[0,2] = 3
print("ORIGIN %%d" %% it.stats().kernel_origin)
''' % os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, ZMC_CACHE_DIR=str(tmp_path))

    def run():
        r = subprocess.run([sys.executable, "-c", script], capture_output=True, text=True, env=env, timeout=300)
        assert r.returncode == 0, r.stderr[-2000:]
        return int([l for l in r.stdout.splitlines() if l.startswith("ORIGIN ")][0].split()[1])

    assert run() == 1                                # compiled by NVRTC, stored
    files = [f for f in os.listdir(tmp_path) if f.endswith(".cubin")]
    assert len(files) == 1
    assert run() == 3                                # another process: from disk
    path = os.path.join(tmp_path, files[0])
    with open(path, "r+b") as f:                     # corrupt the stored key: the file must be ignored and rewritten
        f.seek(20)
        f.write(b"XXXX")
    assert run() == 1
    assert run() == 3
