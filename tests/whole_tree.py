"""Test-side drivers for whole-tree comparisons at sizes one oracle process cannot finish in a test run.

  oracle_tree_fanned        the oracle's tree search with its per-unit sums fanned out over the host cores: orc_unit_sum for every
                            (cell, trial) unit in a process pool, then orc_cell_stats / orc_threshold on the gathered sums, level by level
                            (R5-R7, breadth first). The oracle itself is untouched and is the only arithmetic here; a CPU test pins this
                            driver to oracle.run bit for bit on a small tree (tests/test_oracle_tree.py).
  check_config2_shaped_tree a BASELINE.json configs[1]-shaped run (6-D sin, 4 divisions, depth 3, the paper's rule, no budget) checked as far
                            as its size allows: tiling identity, levels 1-2 cell by cell, the 4e8-cell level 3 by a streamed pass, sampled
                            whole sibling groups and sampled units against the oracle.
"""
import math
import multiprocessing as mp
import os
import time

import numpy as np

import oracle as O
from paper_1902_07916_b200 import workloads as W
from tests import helpers as H


def digits_of(path, k, level):
    out = []
    for _ in range(level):
        out.append(path % k)
        path //= k
    return out[::-1]


def _unit_sums_job(job):
    """Worker: the oracle's per-unit sums S[cell, trial] for a slice of one level's cells (given by their child-index digits)."""
    w, level, cells = job
    cfg = H.oracle_config(w)
    out = np.zeros((len(cells), w.trials))
    for i, digits in enumerate(cells):
        path, coords = O.path_coords(w.dim, w.g, digits)
        for t in range(w.trials):
            out[i, t] = O.unit_sum(cfg, 0, path, level, coords, t)[0]
    return out


def oracle_tree_fanned(w: W.Workload, processes=None, cells_per_job=64) -> O.Result:
    """The oracle's result for a one-instance workload without a budget, as oracle.run(cfg, keep_cells=True) returns it, with the
    sampling spread over `processes` host cores (default: all). Spawned workers: the parent may hold a CUDA context."""
    assert w.n_instances == 1 and w.max_groups_per_level == 0
    k, T, N, L = w.k, w.trials, w.n_samples, w.depth
    prefactor = float(w.params[0][0]) if w.integrand == W.EXP_QUAD else 1.0
    levels, value, var, evals = [], 0.0, 0.0, 0
    parents = [()]
    with mp.get_context("spawn").Pool(processes or os.cpu_count()) as pool:
        for level in range(1, L + 1):
            cells = [p + (j,) for p in parents for j in range(k)]
            jobs = [(w, level, cells[a: a + cells_per_job]) for a in range(0, len(cells), cells_per_job)]
            S = np.concatenate(pool.map(_unit_sums_job, jobs, chunksize=1)) if cells else np.zeros((0, T))
            n = len(cells)
            mu, s, tau = np.zeros(n), np.zeros(n), np.zeros(n)
            paths = []
            for c, digits in enumerate(cells):
                path, coords = O.path_coords(w.dim, w.g, digits)
                paths.append(path)
                V = O.cell_geometry(w.dim, w.lower, w.upper, w.g, level, coords)[2]
                _, mu[c], s[c] = O.cell_stats(S[c], V, prefactor, N)
            for G in range(len(parents)):
                tau[G * k: (G + 1) * k] = O.threshold(s[G * k: (G + 1) * k], w.sigma_multiplier)
            refined = (s > tau) & (level < L)
            value += float(mu[~refined].sum())
            var += float((s[~refined] ** 2).sum())
            evals += n * T * N
            levels.append(O.Level(n, int(refined.sum()), 0, np.zeros(n, dtype=np.uint32), paths, mu, s, tau, refined.astype(np.uint8), S))
            parents = [cells[c] for c in np.nonzero(refined)[0]]
            if not parents:
                break
    return O.Result(np.array([value]), np.array([math.sqrt(var)]), levels, evals)


def check_config2_shaped_tree(w: W.Workload, max_cells_per_level: int, seed: int = 77, groups_in_full: int = 24) -> dict:
    """Run `w` (6-D sin, depth 3, no budget) on the GPU with every level kept and check it; returns a record of the run."""
    import torch
    from paper_1902_07916_b200 import binding as B
    torch.cuda.empty_cache()
    cfg = H.oracle_config(w)
    k, T, N, L = w.k, w.trials, w.n_samples, w.depth
    assert L == 3 and w.max_groups_per_level == 0
    rng = np.random.default_rng(seed)
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=max_cells_per_level)
    t0 = time.perf_counter()
    it.run()
    v, sd = it.result()           # max_cells_per_level == 0: the automatic capacity grows here and the search runs again
    wall = time.perf_counter() - t0
    ws_bytes = it.workspace_bytes()
    st = it.stats()
    assert st.overflow == 0 and st.nonfinite == 0
    lv = [st.level[l] for l in range(L)]
    # ---- tiling invariant: the accepted cells tile the domain
    tiles = sum((lv[l].n_cells - lv[l].n_refined) * k ** (L - 1 - l) for l in range(L))
    assert tiles == k ** L, (tiles, k ** L)
    assert all(lv[l].n_refined == lv[l].n_flagged for l in range(L)) and lv[L - 1].n_flagged == 0      # no budget
    assert all(lv[l + 1].n_cells == lv[l].n_refined * k for l in range(L - 1))
    assert st.total_evals == sum(x.n_cells for x in lv) * T * N
    val, var = 0.0, 0.0
    expect_next = None
    for level in (1, 2):      # T3 on every cell, T2 on sampled units
        gl = it.level_cells(level)
        n = len(gl.mu)
        vol = math.prod((b - a) / w.g ** level for a, b in zip(w.lower, w.upper))
        if level == 1:
            assert gl.path == list(range(k))
        else:
            assert gl.path == [p * k + j for p in expect_next for j in range(k)]
        I = vol * gl.S / float(N)
        mu = I.sum(axis=1) / T
        s = np.sqrt(((I - mu[:, None]) ** 2).sum(axis=1) / T)
        sc = max(np.abs(mu).max(), s.max())
        assert np.abs(gl.mu - mu).max() <= 1e-11 * sc and np.abs(gl.s - s).max() <= 1e-9 * sc
        tau_c, refined, _, _ = H.host_control(gl.mu, gl.s, k, level, L, w.sigma_multiplier, gl.instance.astype(np.int64))
        assert np.abs(gl.tau - tau_c).max() <= 1e-11 * tau_c.max()
        diff = np.nonzero(gl.refined.astype(bool) != refined)[0]
        assert len(diff) == 0 or np.all(np.abs(gl.s[diff] - tau_c[diff]) <= 1e-11 * tau_c[diff])
        refined = gl.refined.astype(bool)
        assert int(refined.sum()) == lv[level - 1].n_refined
        val += float(gl.mu[~refined].sum())
        var += float((gl.s[~refined] ** 2).sum())
        expect_next = [gl.path[i] for i in np.nonzero(refined)[0]]
        for c in rng.integers(0, n, size=8):
            t = int(rng.integers(0, T))
            path, coords = O.path_coords(w.dim, w.g, digits_of(gl.path[c], k, level))
            S_o, _ = O.unit_sum(cfg, 0, path, level, coords, t)
            assert abs(gl.S[c, t] - S_o) <= 1e-12 * N
    # ---- level 3: a streamed pass over every cell (accepted sums), sampled groups in full, sampled units against the oracle
    n3 = lv[2].n_cells
    G3 = n3 // k
    assert G3 == len(expect_next)
    vol3 = math.prod((b - a) / w.g ** 3 for a, b in zip(w.lower, w.upper))
    pick = set(int(g) for g in rng.integers(0, G3, size=groups_in_full)) | {0, G3 - 1}
    groups_per_slab = 512
    sum_mu, sum_var, n_checked_groups = 0.0, 0.0, 0
    for g0 in range(0, G3, groups_per_slab):
        g1 = min(G3, g0 + groups_per_slab)
        if not any(g0 <= g < g1 for g in pick):      # statistics only: cheaper than the identities
            mu, s, ref = it.level_stats_range(3, g0 * k, (g1 - g0) * k)
            assert not ref.any()
            sum_mu += float(mu.sum())
            sum_var += float((s ** 2).sum())
            continue
        sl = it.level_cells_range(3, g0 * k, (g1 - g0) * k)
        assert not sl.refined.any()
        sum_mu += float(sl.mu.sum())
        sum_var += float((sl.s ** 2).sum())
        for g in sorted(p for p in pick if g0 <= p < g1):
            a = (g - g0) * k
            assert sl.path[a: a + k] == [expect_next[g] * k + j for j in range(k)]
            Sg = sl.S[a: a + k]
            I = vol3 * Sg / float(N)
            mu = I.sum(axis=1) / T
            s = np.sqrt(((I - mu[:, None]) ** 2).sum(axis=1) / T)
            sc = max(np.abs(mu).max(), s.max())
            assert np.abs(sl.mu[a: a + k] - mu).max() <= 1e-11 * sc and np.abs(sl.s[a: a + k] - s).max() <= 1e-9 * sc
            tau = s.mean() + w.sigma_multiplier * np.sqrt(((s - s.mean()) ** 2).mean())
            assert np.abs(sl.tau[a: a + k] - tau).max() <= 1e-9 * tau
            n_checked_groups += 1
            for j in rng.integers(0, k, size=2):      # T2 at level 3
                t = int(rng.integers(0, T))
                path, coords = O.path_coords(w.dim, w.g, digits_of(sl.path[a + j], k, 3))
                S_o, _ = O.unit_sum(cfg, 0, path, 3, coords, t)
                assert abs(Sg[j, t] - S_o) <= 1e-12 * N
    assert n_checked_groups == len(pick)
    val += sum_mu
    var += sum_var
    assert abs(v[0] - val) <= 1e-9 * max(abs(val), math.sqrt(var))      # numpy's pairwise sums over 4e8 cells vs the device's fixed tree
    assert abs(sd[0] - math.sqrt(var)) <= 1e-9 * math.sqrt(var)
    closed = H.closed_sin_sum(w.lower, w.upper)
    assert abs(v[0] - closed) <= 4 * sd[0]
    z = (v[0] - closed) / (sd[0] / math.sqrt(T - 1))
    rec = {"workload": "%s: 6-D sin, g = %d, N = %d, T = %d, depth 3, m = %g, no budget" % (w.name, w.g, N, T, w.sigma_multiplier),
           "value": float(v[0]), "std": float(sd[0]), "closed_form": closed, "z_vs_std_over_sqrt_T_minus_1": z,
           "cells_per_level": [int(x.n_cells) for x in lv], "flagged_per_level": [int(x.n_flagged) for x in lv],
           "work_items_level3": int(lv[2].n_cells) * T,
           "evals": int(st.total_evals), "device_ms": float(st.total_ms), "wall_s_run_plus_result": wall,
           "evals_per_s": st.total_evals / (st.total_ms * 1e-3),
           "sample_ms_per_level": [float(x.sample_ms) for x in lv], "control_ms_per_level": [float(x.control_ms) for x in lv],
           "workspace_bytes": int(ws_bytes), "max_cells_per_level": int(max_cells_per_level) or "automatic (grown by zmc_result)", "level3_groups_checked_in_full": n_checked_groups}
    it.close()
    return rec
