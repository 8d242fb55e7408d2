"""GPU tests of boundary behaviour added in round 2 (include/zmc.h): zmc_set_option validates before it changes anything,
zmc_level_cells_range, the compile-at-call contract of zmc_set_integrand_source, and the largest-spread budget when the
threshold is negative (sigma_multiplier < 0 flags cells whose spread is exactly zero)."""
import numpy as np
import pytest

import oracle as O
from paper_1902_07916_b200 import binding as B
from paper_1902_07916_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu


def test_rejected_option_leaves_a_caller_owned_workspace_usable():
    """A caller-owned workspace fixes the layout. An option that would change it is refused with ZMC_ERR_STATE and the
    context keeps its old value: the next run is bit-identical to the first (it used to keep the new value with the old layout:
    out-of-bounds partial sums, a null partial_q or null piv/quota on the next run)."""
    w = W.config1()
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 12)
    it.use_torch_workspace()
    it.run()
    v0, s0 = it.result()
    S0 = it.level_cells(2).S.copy()
    for key, val in ((B.OPT_TARGET_ITEMS, 1 << 20), (B.OPT_SPREAD, B.SPREAD_SAMPLES), (B.OPT_BUDGET_ORDER, B.BUDGET_LARGEST_SPREAD),
                     (B.OPT_KEEP_LEVEL_STATS, 0), (B.OPT_MAX_CELLS_PER_LEVEL, 1 << 16)):
        with pytest.raises(B.ZmcError) as e:
            it.set_option(key, val)
        assert e.value.status == B.ERR_STATE, key
        it.set_option(B.OPT_MAX_GROUPS_PER_LEVEL, 7)        # a budget that binds nothing here (5 flagged); allowed: no layout change
        it.run()
        v, s = it.result()
        assert v[0] == v0[0] and s[0] == s0[0]
        np.testing.assert_array_equal(it.level_cells(2).S, S0)
    with pytest.raises(B.ZmcError) as e:
        it.set_option(B.OPT_TARGET_ITEMS, 0)                # invalid values are ZMC_ERR_ARG as before
    assert e.value.status == B.ERR_ARG
    # the documented way out: set the option after giving the workspace back, then provide one of the new size
    it.set_workspace((it._ws.data_ptr() + 255) & ~255, it._ws.numel() - 256)      # same memory: resets the layout
    it.set_option(B.OPT_TARGET_ITEMS, 320)
    it.use_torch_workspace()
    it.run()
    v, s = it.result()
    assert abs(v[0] - v0[0]) <= 1e-12 * abs(v0[0])
    it.close()


def test_level_cells_range_matches_the_full_dump():
    w = W.config2().with_(n_samples=64, depth=2, max_groups_per_level=3)
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 16)
    it.run()
    it.result()
    full = it.level_cells(2)
    n = len(full.mu)
    assert n == 3 * w.k
    for first, count in ((0, n), (0, 1), (n - 1, 1), (w.k - 3, 7), (2 * w.k + 5, 100), (17, 0)):
        r = it.level_cells_range(2, first, count)
        sl = slice(first, first + count)
        np.testing.assert_array_equal(r.mu, full.mu[sl])
        np.testing.assert_array_equal(r.s, full.s[sl])
        np.testing.assert_array_equal(r.tau, full.tau[sl])
        np.testing.assert_array_equal(r.S, full.S[sl])
        np.testing.assert_array_equal(r.refined, full.refined[sl])
        np.testing.assert_array_equal(r.instance, full.instance[sl])
        assert r.path == full.path[sl]
    for first, count in ((n, 1), (n - 1, 2), (0, n + 1)):
        with pytest.raises(B.ZmcError) as e:
            it.level_cells_range(2, first, count)
        assert e.value.status == B.ERR_ARG
    it.close()


FLOAT_ONLY = "__device__ float only_f(const float* x, int dim, const float* p, int np) { return p[0] * x[0] + x[1]; }"


def test_user_source_is_compiled_at_the_call_for_the_precision_in_force():
    """include/zmc.h: a source with one overload needs that precision set BEFORE zmc_set_integrand_source; a later
    precision change that cannot compile returns ZMC_ERR_COMPILE and keeps the working setting."""
    mk = lambda: B.Integrator(2, [0.0, 0.0], [1.0, 2.0], 3, 500, 4, 2, 1.5, 5)
    it = mk()
    with pytest.raises(B.ZmcError) as e:                      # default precision is F64: the double overload is missing
        it.set_integrand_source(FLOAT_ONLY, "only_f", np.array([[3.0]]), 1)
    assert e.value.status == B.ERR_COMPILE
    it.close()
    it = mk()
    it.set_option(B.OPT_PRECISION, B.F32)
    it.set_integrand_source(FLOAT_ONLY, "only_f", np.array([[3.0]]), 1)
    it.run()
    v, s = it.result()
    closed = 2.0 * (3.0 * 0.5 + 1.0)                         # int (3 x0 + x1) over [0,1]x[0,2]
    assert abs(v[0] - closed) <= 4 * s[0] + 1e-6
    with pytest.raises(B.ZmcError) as e:
        it.set_option(B.OPT_PRECISION, B.F64)
    assert e.value.status == B.ERR_COMPILE
    it.run()                                                  # still the FP32 program
    v2, s2 = it.result()
    assert v2[0] == v[0] and s2[0] == s[0]
    it.close()


@pytest.mark.parametrize("budget", [2, 1000])
def test_largest_spread_budget_with_negative_threshold(budget):
    """sigma_multiplier < 0 on a narrow Gaussian: most cells have s == +0 exactly and tau < 0, so they are flagged with key 0.
    With a budget that does not bind (1000) every one of them must be refined, as the oracle does (they used to be dropped by a
    zero tie quota, leaving unwritten parent slots); with a binding budget the largest spreads win and zeros come last."""
    w = W.Workload("g2neg", 2, (-1.0, -1.0), (1.0, 1.0), 5, 200, 4, 2, -0.5, 21, W.EXP_QUAD, W.F32,
                   params=W.gaussian_params(2, 0.01), max_groups_per_level=budget)
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 16, budget_order=B.BUDGET_LARGEST_SPREAD)
    it.run()
    ores = O.run(H.oracle_config(w, budget_order=O.BUDGET_LARGEST_SPREAD), keep_cells=True)
    l1 = ores.levels[0]
    assert (l1.s == 0.0).sum() >= 10 and l1.tau[0] < 0.0          # the case is what it claims to be
    if budget == 1000:
        assert l1.n_refined == 25                                  # s >= 0 > tau everywhere
    H.compare_tree(it, ores, w)
    it.close()
