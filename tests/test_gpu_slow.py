"""BASELINE.json configs[1] WHOLE, once, under the paper's rule ("until ... all ... are lower than the threshold
or the maximal partition depth is reached"): 6-D sin, 4 divisions per axis, 1e5 samples, 5 trials, depth 3, m = 1.5, no
refinement budget -- about 2e14 integrand evaluations, 4e8 level-3 cells, ~13 minutes on one B200, ~110 GB of workspace with the
per-level arrays kept (max_cells_per_level = 2^29). Far beyond the driver's 20-minute pytest step, so it runs only when asked:

    ZMC_RUN_SLOW=1 python -m pytest tests/test_gpu_slow.py -m gpu -s

Checked at that size (the oracle cannot run it whole):
  * tiling: sum_l n_accepted(l) * k^(L-l) = k^L from zmc_stats (the accepted cells tile the domain);
  * levels 1-2: T3 -- every cell's (mu, s) from the dumped sums, tau, flags, compaction output re-derived in numpy;
  * level 3: T2 -- sampled (cell, trial) units recomputed by the oracle; T3 on sampled whole sibling groups (zmc_level_cells_range),
    identities = children of the expected parents; the level's accepted sums from a streamed pass over all 4e8 cells;
  * all levels: sampled units against the oracle;
  * result within 4 sigma of the closed form; the z-score against std/sqrt(T-1) is printed.
A JSON summary goes to gpurun_out/r2_cfg2_whole.json (profiles/r2_cfg2_whole.md quotes it).

Second slow test: BASELINE.json configs[2] (9-D narrow Gaussian) whole on BOTH sides -- the oracle's complete tree on one host core
(~9 minutes) against the GPU's, all 78 732 cells (-k config3).
"""
import json
import math
import os
import time

import numpy as np
import pytest

import oracle as O
from paper_1902_07916_b200 import binding as B
from paper_1902_07916_b200 import workloads as W
from tests import helpers as H

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _digits(path, k, level):
    out = []
    for _ in range(level):
        out.append(path % k)
        path //= k
    return out[::-1]


@pytest.mark.skipif(os.environ.get("ZMC_RUN_SLOW") != "1", reason="~13 GPU-minutes; set ZMC_RUN_SLOW=1")
def test_config2_whole_under_the_papers_rule():
    w = W.config2(depth=3, budget=0)
    cfg = H.oracle_config(w)
    k, T, N, L = w.k, w.trials, w.n_samples, w.depth
    rng = np.random.default_rng(77)
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=1 << 29)
    ws_bytes = it.workspace_bytes()
    t0 = time.perf_counter()
    it.run()
    v, sd = it.result()
    wall = time.perf_counter() - t0
    st = it.stats()
    assert st.overflow == 0 and st.nonfinite == 0
    lv = [st.level[l] for l in range(L)]
    # ---- tiling invariant
    tiles = sum((lv[l].n_cells - lv[l].n_refined) * k ** (L - 1 - l) for l in range(L))
    assert tiles == k ** L, (tiles, k ** L)
    assert all(lv[l].n_refined == lv[l].n_flagged for l in range(L)) and lv[L - 1].n_flagged == 0      # no budget
    assert all(lv[l + 1].n_cells == lv[l].n_refined * k for l in range(L - 1))
    assert st.total_evals == sum(x.n_cells for x in lv) * T * N
    val, var = 0.0, 0.0
    expect_next = None
    for level in (1, 2):
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
        tau_c, refined, a_val, a_var = H.host_control(gl.mu, gl.s, k, level, L, w.sigma_multiplier, gl.instance.astype(np.int64))
        assert np.abs(gl.tau - tau_c).max() <= 1e-11 * tau_c.max()
        diff = np.nonzero(gl.refined.astype(bool) != refined)[0]
        assert len(diff) == 0 or np.all(np.abs(gl.s[diff] - tau_c[diff]) <= 1e-11 * tau_c[diff])
        refined = gl.refined.astype(bool)
        assert int(refined.sum()) == lv[level - 1].n_refined
        val += float(gl.mu[~refined].sum())
        var += float((gl.s[~refined] ** 2).sum())
        expect_next = [gl.path[i] for i in np.nonzero(refined)[0]]
        for c in rng.integers(0, n, size=8):       # T2
            t = int(rng.integers(0, T))
            path, coords = O.path_coords(w.dim, w.g, _digits(gl.path[c], k, level))
            S_o, _ = O.unit_sum(cfg, 0, path, level, coords, t)
            assert abs(gl.S[c, t] - S_o) <= 1e-12 * N
    # ---- level 3: streamed pass over every cell (accepted sums), sampled groups in full, sampled units against the oracle
    n3 = lv[2].n_cells
    G3 = n3 // k
    assert G3 == len(expect_next)
    vol3 = math.prod((b - a) / w.g ** 3 for a, b in zip(w.lower, w.upper))
    pick = set(int(g) for g in rng.integers(0, G3, size=24)) | {0, G3 - 1}
    groups_per_slab = 512
    sum_mu, sum_var, n_checked_groups = 0.0, 0.0, 0
    for g0 in range(0, G3, groups_per_slab):
        g1 = min(G3, g0 + groups_per_slab)
        sl = it.level_cells_range(3, g0 * k, (g1 - g0) * k) if any(g0 <= g < g1 for g in pick) else None
        if sl is None:      # statistics only: cheaper than the identities
            cnt = (g1 - g0) * k
            mu = np.zeros(cnt)
            s = np.zeros(cnt)
            ref = np.zeros(cnt, dtype=np.uint8)
            it._check(it._L.zmc_level_cells_range(it._h, 3, g0 * k, cnt, None, None, None, B._dp(mu), B._dp(s), None,
                                                  B._ptr(ref, B.C.c_uint8), None))
            assert not ref.any()
            sum_mu += float(mu.sum())
            sum_var += float((s ** 2).sum())
            continue
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
                path, coords = O.path_coords(w.dim, w.g, _digits(sl.path[a + j], k, 3))
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
    out = {"workload": "cfg2_sin6d (BASELINE.json configs[1], depth 3, no budget)", "value": float(v[0]), "std": float(sd[0]),
           "closed_form": closed, "z_vs_std_over_sqrt_T_minus_1": z,
           "cells_per_level": [int(x.n_cells) for x in lv], "flagged_per_level": [int(x.n_flagged) for x in lv],
           "evals": int(st.total_evals), "device_ms": float(st.total_ms), "wall_s_run_plus_result": wall,
           "evals_per_s": st.total_evals / (st.total_ms * 1e-3),
           "sample_ms_per_level": [float(x.sample_ms) for x in lv], "control_ms_per_level": [float(x.control_ms) for x in lv],
           "workspace_bytes": int(ws_bytes), "max_cells_per_level": 1 << 29, "level3_groups_checked_in_full": n_checked_groups}
    print(json.dumps(out))
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    json.dump(out, open(os.path.join(ROOT, "gpurun_out", "r2_cfg2_whole.json"), "w"), indent=1)
    it.close()


@pytest.mark.skipif(os.environ.get("ZMC_RUN_SLOW") != "1", reason="~7 minutes of the oracle on one host core; set ZMC_RUN_SLOW=1")
def test_config3_whole_gpu_against_the_oracle_whole():
    """BASELINE.json configs[2] WHOLE on both sides: the 9-D narrow Gaussian, 4 levels x 19 683 cells, 7.87e9 evaluations. The oracle
    runs the complete tree on one host core (~6 minutes: its time-to-result, measured, not extrapolated) and every one of the 78 732
    cells is compared -- per-(cell, trial) sums, (mu, s), tau, refined sets, cell identities -- plus the result. Run it alone:

        ZMC_RUN_SLOW=1 python -m pytest tests/test_gpu_slow.py -m gpu -s -k config3
    """
    w = W.config3()
    it = B.from_workload(w, keep_level_stats=True, max_cells_per_level=w.max_cells_per_level)
    it.run()
    v, s = it.result()
    st = it.stats()
    t0 = time.perf_counter()
    ores = O.run(H.oracle_config(w), keep_cells=True)
    oracle_s = time.perf_counter() - t0
    n = H.compare_tree(it, ores, w)
    assert n == 4 * 19683
    closed = H.closed_exp_quad(w.params[0], w.lower, w.upper)
    assert abs(v[0] - closed) <= 4 * s[0]
    rec = {"workload": "cfg3_gauss9d (BASELINE.json configs[2], whole)", "cells_compared": n, "value_gpu": float(v[0]), "std_gpu": float(s[0]),
           "value_oracle": float(ores.value[0]), "std_oracle": float(ores.std[0]), "closed_form": closed,
           "evals": int(st.total_evals), "gpu_device_ms": float(st.total_ms), "oracle_seconds_one_core": oracle_s,
           "oracle_evals_per_s": st.total_evals / oracle_s, "refined_per_level": [int(st.level[l].n_refined) for l in range(4)]}
    print(json.dumps(rec))
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    with open(os.path.join(ROOT, "gpurun_out", "r2_cfg3_whole_vs_oracle.json"), "w") as f:
        json.dump(rec, f, indent=1)
    it.close()
