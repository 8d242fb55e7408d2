"""The single-launch path (ZMC_OPT_SINGLE_LAUNCH, csrc/zmc_tree.cuh): one cooperative kernel for the whole tree search gives the
same bits as the multi-launch path -- every per-(cell, trial) sum, (mu, s, tau), refined set and result -- on small trees
(one block takes a sibling group through statistics, threshold and count), on sibling groups of several control tiles (the
step-by-step order with grid barriers), with instances and a budget, on trees that end early; and it still matches the oracle."""
import numpy as np
import pytest

import oracle as O
from paper_1902_07916_b200 import binding as B, workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _pair(w, **kw):
    out = []
    for single in (0, 1):
        it = B.from_workload(w, keep_level_stats=True, single_launch=single, **kw)
        it.run()
        out.append(it)
    return out


def _same_bits(a, b, depth):
    sa, sb = a.stats(), b.stats()
    assert sa.kernel_launches > 1 and sb.kernel_launches == 1
    for lev in range(1, depth + 1):
        assert sa.level[lev - 1].n_cells == sb.level[lev - 1].n_cells
        assert sa.level[lev - 1].n_flagged == sb.level[lev - 1].n_flagged
        assert sa.level[lev - 1].n_refined == sb.level[lev - 1].n_refined
        if sa.level[lev - 1].n_cells == 0:
            continue
        la, lb = a.level_cells(lev), b.level_cells(lev)
        assert la.path == lb.path
        for f in ("instance", "S", "mu", "s", "tau", "refined"):
            np.testing.assert_array_equal(getattr(la, f), getattr(lb, f), err_msg="level %d %s" % (lev, f))
    va, da = a.result()
    vb, db = b.result()
    np.testing.assert_array_equal(va, vb)
    np.testing.assert_array_equal(da, db)


def test_config1_single_launch_is_bit_identical_and_matches_the_oracle():
    w = W.config1()
    a, b = _pair(w)
    _same_bits(a, b, w.depth)
    ores = O.run(H.oracle_config(w), keep_cells=True)
    assert H.compare_tree(b, ores, w) == 384
    # default = auto: this problem (6.4e5 evaluations at level 1) takes the single launch
    c = B.from_workload(w)
    c.run()
    assert c.stats().kernel_launches == 1
    np.testing.assert_array_equal(c.result()[0], b.result()[0])
    b.run()                                             # re-run on the same context
    np.testing.assert_array_equal(c.result()[0], b.result()[0])
    for it in (a, b, c):
        it.close()


def test_auto_keeps_large_problems_on_the_multi_launch_path():
    w = W.config2(depth=2, budget=1).with_(n_samples=2000)        # 4096 * 5 * 2000 = 4.1e7 evaluations at level 1
    it = B.from_workload(w, max_cells_per_level=4096)
    it.run()
    st = it.stats()
    assert st.kernel_launches == 2 + 6 * 2
    it.close()


def test_auto_looks_at_the_later_levels_too():
    """Auto takes the single launch only if no LATER level can outgrow the small first one by much: a deep tree without a budget may
    grow to the level capacity (kernel by kernel), the same tree with a budget of 4 parents per level cannot (one launch)."""
    w = W.Workload("s2_deep", 2, (0.0, 0.0), (7.0, 5.0), 5, 64, 5, 6, 0.3, 9, W.SIN_SUM, W.F64)
    it = B.from_workload(w)
    it.run()
    free = (it.stats().kernel_launches, it.result())
    it.close()
    it = B.from_workload(w.with_(max_groups_per_level=4))
    it.run()
    capped = it.stats().kernel_launches
    it.close()
    assert free[0] == 2 + 6 * 6 and capped == 1
    it = B.from_workload(w, single_launch=1)              # the preference still overrides auto, with the same bits
    it.run()
    assert it.stats().kernel_launches == 1
    np.testing.assert_array_equal(it.result()[0], free[1][0])
    it.close()


def test_refused_cooperative_launch_falls_back_to_the_multi_launch_path(monkeypatch):
    """A cooperative launch can be refused where plain launches work (MPS thread percentage, green contexts, tools in between).
    ZMC_DEBUG_REFUSE_COOPERATIVE=1 makes the library take that branch: zmc_run then goes kernel by kernel, with the same bits, under
    'whenever possible' and under auto; a context created afterwards, without the variable, takes the single launch again."""
    w = W.config1()
    ref = B.from_workload(w, single_launch=0)
    ref.run()
    v0, s0 = ref.result()
    ref.close()
    monkeypatch.setenv("ZMC_DEBUG_REFUSE_COOPERATIVE", "1")
    for single in (1, 2):
        it = B.from_workload(w, single_launch=single)
        for _ in range(2):                                  # the second run does not try the cooperative launch again
            it.run()
            assert it.stats().kernel_launches == 2 + 6 * 2
            v, s = it.result()
            np.testing.assert_array_equal(v, v0)
            np.testing.assert_array_equal(s, s0)
        it.close()
    monkeypatch.delenv("ZMC_DEBUG_REFUSE_COOPERATIVE")
    it = B.from_workload(w)
    it.run()
    assert it.stats().kernel_launches == 1
    np.testing.assert_array_equal(it.result()[0], v0)
    it.close()


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_batched_instances_with_budget(precision):
    w = W.config4(n_instances=37).with_(g=3, n_samples=515, depth=3, max_groups_per_level=2, precision=precision)
    a, b = _pair(w, max_cells_per_level=37 * 81 * 2)
    _same_bits(a, b, 3)
    ores = O.run(H.oracle_config(w), keep_cells=True)
    H.compare_tree(b, ores, w)
    a.close(); b.close()


def test_three_tiles_per_group():
    """k = 100^2 = 10000 cells: three 4096-cell control tiles per sibling group (the three-pass threshold, a grid barrier between
    the passes)."""
    w = W.Workload("solo_limit", 2, (0.0, 0.0), (10.0, 7.0), 100, 96, 3, 2, 1.0, 17, W.SIN_SUM, W.F32, max_groups_per_level=2)
    a, b = _pair(w, max_cells_per_level=2 * 10000)
    _same_bits(a, b, 2)
    assert b.stats().level[1].n_cells == 20000
    ores = O.run(H.oracle_config(w), keep_cells=True)
    H.compare_tree(b, ores, w)
    a.close(); b.close()


def test_two_tiles_per_group_and_empty_levels():
    """k = 70^2 = 4900 (two control tiles); a constant integrand flags nothing: levels 2 and 3 are empty."""
    w = W.Workload("tiles_solo", 2, (0.0, 0.0), (1.0, 1.0), 70, 33, 4, 2, 0.5, 3, W.EXP_QUAD, W.F32,
                   params=np.array([[1.0, 30.0, 0.4, 0.6]]), max_groups_per_level=1)
    a, b = _pair(w, max_cells_per_level=4900)
    _same_bits(a, b, 2)
    a.close(); b.close()
    w = W.Workload("const", 3, (0.0,) * 3, (1.0,) * 3, 3, 100, 3, 3, 1.0, 1, W.CONST, W.F64, params=np.array([[2.5]]))
    a, b = _pair(w)
    _same_bits(a, b, 3)
    v, s = b.result()
    assert abs(v[0] - 2.5) < 1e-12 and b.stats().level[1].n_cells == 0
    a.close(); b.close()


def test_forced_single_launch_where_it_does_not_exist_falls_back():
    """R13 (sum-of-squares kernel) and user integrands have no tree kernel: the option is a preference, the run still works."""
    w = W.config1()
    it = B.from_workload(w, single_launch=1, spread=B.SPREAD_SAMPLES)
    it.run()
    assert it.stats().kernel_launches > 1
    it.close()


def test_depth_one_and_high_dimension_fp64():
    """Depth 1 (the first level is the last: no scan, no compaction); D = 7 in FP64 (the one-block-per-SM instance of the tree
    kernel) -- each bit-identical to its multi-launch run."""
    w = W.config1().with_(depth=1)
    a, b = _pair(w)
    _same_bits(a, b, 1)
    ores = O.run(H.oracle_config(w), keep_cells=True)
    H.compare_tree(b, ores, w)
    a.close(); b.close()
    w = W.Workload("d7_f64", 7, (0.0,) * 7, (1.0,) * 7, 2, 301, 3, 3, 0.5, 23, W.EXP_QUAD, W.F64,
                   params=np.array([[1.0, 9.0] + [0.4] * 7]), max_groups_per_level=3)
    a, b = _pair(w, max_cells_per_level=3 * 128)
    _same_bits(a, b, 3)
    ores = O.run(H.oracle_config(w), keep_cells=True)
    H.compare_tree(b, ores, w)                         # FP64 exp: libdevice vs libm, <= 4 ulp per value of at most 1: 1e-15 * N, inside the rule's 1e-12 * N
    a.close(); b.close()
    # fast math and D > 8 have no tree kernel: the option is a preference, the run takes the multi-launch path
    w = W.config2(depth=2, budget=2).with_(n_samples=150)
    it = B.from_workload(w, max_cells_per_level=2 * 4096, math=B.MATH_FAST, single_launch=1)
    it.run()
    assert it.stats().kernel_launches > 1
    it.close()
