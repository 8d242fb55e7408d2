"""Whole trees at BASELINE.json's sizes inside the default `-m gpu` run (the driver's GPU test step), where round 2 had them as slow tests:

  configs[2] whole on BOTH sides    the 9-D narrow Gaussian, 4 levels x 19 683 cells: the oracle's complete tree, its 393 660 per-unit sums
                                    fanned out over the host cores (7.87e9 evaluations), against the GPU's, all 78 732 cells;
  configs[1]-shaped, N = 8          the same D, g, T, m, depth 3 and the paper's rule (no budget) as configs[1], with 8 samples per unit:
                                    306 -> 108 142 refined cells -> a level 3 of 4.43e8 cells (configs[1] itself: 309 -> 109 781 -> 4.50e8):
                                    PAPER.md:73's "until ... the maximal partition depth is reached" at full width, 113 GB of kept arrays;
  work items beyond 2^32            a level of 4.59e9 (cell, trial) work items: the 64-bit branch of the item decoding (zmc_divmod,
                                    ZmcUnit::decode) and 64-bit indices in the statistics kernels, which no other test reaches.
The real-N configs[1] run (14 GPU-minutes) stays in tests/test_gpu_slow.py.
"""
import math
import os
import time

import numpy as np
import pytest

import oracle as O
from paper_1902_07916_b200 import binding as B, workloads as W
from tests import helpers as H, whole_tree as WT

pytestmark = pytest.mark.gpu


def test_config3_whole_gpu_against_the_oracle_whole():
    w = W.config3()
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=w.max_cells_per_level)
    it.run()
    v, s = it.result()
    t0 = time.perf_counter()
    ores = WT.oracle_tree_fanned(w)
    oracle_s = time.perf_counter() - t0
    n = H.compare_tree(it, ores, w)
    assert n == 4 * 19683
    assert [l.n_refined for l in ores.levels] == [1, 1, 1, 0]
    closed = H.closed_exp_quad(w.params[0], w.lower, w.upper)
    assert abs(v[0] - closed) <= 4 * s[0]
    print("cfg3 whole: %d cells compared; oracle over %d cores %.1f s; value %.9f +- %.6f (oracle %.9f)" %
          (n, os.cpu_count(), oracle_s, v[0], s[0], ores.value[0]))
    it.close()


def test_config2_shaped_tree_with_a_4e8_cell_level():
    w = W.config2(depth=3, budget=0).with_(n_samples=8)
    rec = WT.check_config2_shaped_tree(w, 1 << 29)
    assert rec["cells_per_level"] == [4096, 306 * 4096, 108142 * 4096]      # what the oracle gives for levels 1 and 2 (depth-2 run)
    print("cfg2-shaped N=8:", rec)


def test_work_items_beyond_2_32():
    """6-D sin, 8 divisions per axis (k = 262 144), T = 250 trials, N = 2, depth 2 with a budget of 70 refined cells: level 2 has exactly
    70 * 262 144 = 1.835e7 cells = 4.59e9 (cell, trial) work items -- item indices pass 2^32 at cell 17 179 869. Sampled units on both
    sides of that index and at the very end against the oracle, statistics of those cells re-derived from the dumped sums, identities from
    the expected parents, the level's accepted sums by a streamed pass. 110 GB of workspace."""
    import torch
    torch.cuda.empty_cache()
    budget = 70
    w = W.Workload("sin6_items_2p32", 6, (0.0,) * 6, (10.0,) * 6, 8, 2, 250, 2, 1.0, 41, W.SIN_SUM, W.F32, max_groups_per_level=budget)
    cfg = H.oracle_config(w)
    k, T, N = w.k, w.trials, w.n_samples
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=budget * k)
    it.run()
    v, sd = it.result()
    st = it.stats()
    assert st.overflow == 0 and st.nonfinite == 0
    n2 = st.level[1].n_cells
    assert st.level[0].n_cells == k and st.level[0].n_refined == budget < st.level[0].n_flagged and n2 == budget * k
    assert n2 * T > 2 ** 32
    rng = np.random.default_rng(9)
    # ---- level 1: every cell (T3), the first 70 flagged cells in path order are the parents (R12)
    g1 = it.level_cells(1)
    vol1 = math.prod((b - a) / w.g for a, b in zip(w.lower, w.upper))
    I = vol1 * g1.S / float(N)
    mu = I.sum(axis=1) / T
    s = np.sqrt(((I - mu[:, None]) ** 2).sum(axis=1) / T)
    sc = max(np.abs(mu).max(), s.max())
    assert np.abs(g1.mu - mu).max() <= 1e-11 * sc and np.abs(g1.s - s).max() <= 1e-9 * sc
    _, refined, _, _ = H.host_control(g1.mu, g1.s, k, 1, 2, w.sigma_multiplier, np.zeros(k, dtype=np.int64), budget=budget)
    np.testing.assert_array_equal(g1.refined.astype(bool), refined)
    parents = [g1.path[i] for i in np.nonzero(refined)[0]]
    val = float(g1.mu[~refined].sum())
    var = float((g1.s[~refined] ** 2).sum())
    # ---- level 2: ranges at the start, across the 2^32-th work item, at the end, and three random ones
    vol2 = vol1 / w.g ** w.dim
    edge = 2 ** 32 // T
    count = 512
    firsts = [0, edge - count // 2, n2 - count] + [int(x) for x in rng.integers(0, n2 - count, size=3)]
    n_units = 0
    for first in firsts:
        sl = it.level_cells_range(2, first, count)
        cells = np.arange(first, first + count)
        assert sl.path == [parents[c // k] * k + c % k for c in cells]
        I = vol2 * sl.S / float(N)
        mu = I.sum(axis=1) / T
        s = np.sqrt(((I - mu[:, None]) ** 2).sum(axis=1) / T)
        sc = max(np.abs(mu).max(), s.max())
        assert np.abs(sl.mu - mu).max() <= 1e-11 * sc and np.abs(sl.s - s).max() <= 1e-9 * sc
        assert not sl.refined.any()
        for i in list(rng.integers(0, count, size=6)) + [count // 2 - 1, count // 2]:
            for t in (0, int(rng.integers(0, T)), T - 1):
                path, coords = O.path_coords(w.dim, w.g, WT.digits_of(sl.path[i], k, 2))
                S_o, _ = O.unit_sum(cfg, 0, path, 2, coords, t)
                assert abs(sl.S[i, t] - S_o) <= 1e-12 * N, (first, i, t)
                n_units += 1
    # ---- the level's accepted sums, streamed
    slab = 1 << 21
    for first in range(0, n2, slab):
        mu, s, ref = it.level_stats_range(2, first, min(slab, n2 - first))
        assert not ref.any()
        val += float(mu.sum())
        var += float((s ** 2).sum())
    assert abs(v[0] - val) <= 1e-9 * max(abs(val), math.sqrt(var))
    assert abs(sd[0] - math.sqrt(var)) <= 1e-9 * math.sqrt(var)
    closed = H.closed_sin_sum(w.lower, w.upper)
    assert abs(v[0] - closed) <= 4 * sd[0]
    print("items > 2^32: level 2 has %d cells = %.3e work items; %d units against the oracle; level-2 sampling %.1f ms, control %.1f ms" %
          (n2, n2 * T, n_units, st.level[1].sample_ms, st.level[1].control_ms))
    it.close()


def test_automatic_capacity_grows_to_what_the_tree_needs():
    """BASELINE.json configs[1] as given must run through zmc_create / zmc_set_integrand / zmc_run / zmc_result with NO option set. Its
    level 3 has 4.5e8 cells, far beyond the first automatic guess (2^22): the search stops at the overflow, zmc_result reads what level 3
    needed, re-allocates and runs again. Here on the N = 8 tree of the same shape (4.43e8 cells): same bits as a run that was given the
    room up front, the level sizes of the kept-array test above, and a workspace sized to the need. A caller-owned workspace cannot
    grow: ZMC_ERR_CAPACITY with the need in the message."""
    import torch
    torch.cuda.empty_cache()
    w = W.config2(depth=3, budget=0).with_(n_samples=8)
    it = B.from_workload(w)                                   # precision and math mode only
    it.run()
    v, s = it.result()                                        # grows and re-runs inside
    st = it.stats()
    assert st.overflow == 0
    assert [st.level[l].n_cells for l in range(3)] == [4096, 306 * 4096, 108142 * 4096]
    grown = it.workspace_bytes()
    it.close()
    assert grown < 32 * 2 ** 30                               # 4.43e8 * (1 + 1/16) cells, 56 bytes each
    ref = B.from_workload(w, max_cells_per_level=108142 * 4096)
    ref.run()
    v0, s0 = ref.result()
    ref.close()
    np.testing.assert_array_equal(v, v0)
    np.testing.assert_array_equal(s, s0)
    # a workspace the caller owns is a hard limit
    it = B.from_workload(w)
    it.use_torch_workspace()
    it.run()
    with pytest.raises(B.ZmcError) as e:
        it.result()
    assert e.value.status == B.ERR_CAPACITY and "level 3 needed 442949632 cells" in str(e.value), str(e.value)
    it.close()
    torch.cuda.empty_cache()
