"""Test helpers: closed forms (independent of oracle/ and of the CUDA path) and
Workload -> oracle.Config conversion."""
import math

import mpmath as mp
import numpy as np

import oracle as O
from paper_1902_07916_b200 import workloads as W

def oracle_config(w: W.Workload, **over) -> O.Config:
    return O.config_from_workload(w, **over)


def closed_sin_sum(lower, upper) -> float:
    """Integral of sin(sum x_d) over a box = Im prod_d (e^{i b_d} - e^{i a_d}) / i  (BASELINE.json north_star)."""
    mp.mp.dps = 40
    z = mp.mpc(1)
    for a, b in zip(lower, upper):
        z *= (mp.expj(b) - mp.expj(a)) / mp.mpc(0, 1)
    return float(z.imag)


def closed_exp_quad(params, lower, upper) -> float:
    """Integral of A exp(-a |x-c|^2) over a box = A prod_d sqrt(pi/a)/2 [erf(sqrt a (b_d-c_d)) - erf(sqrt a (a_d-c_d))]."""
    mp.mp.dps = 40
    A, a = mp.mpf(float(params[0])), mp.mpf(float(params[1]))
    v = A
    for d, (lo, hi) in enumerate(zip(lower, upper)):
        c = mp.mpf(float(params[2 + d]))
        v *= mp.sqrt(mp.pi / a) / 2 * (mp.erf(mp.sqrt(a) * (hi - c)) - mp.erf(mp.sqrt(a) * (lo - c)))
    return float(v)


def closed_linear(params, lower, upper) -> float:
    vol = math.prod(b - a for a, b in zip(lower, upper))
    return vol * (params[0] + sum(params[1 + d] * 0.5 * (a + b) for d, (a, b) in enumerate(zip(lower, upper))))


def var_sin_sum_box(lower, upper) -> float:
    """Variance of f = sin(sum x) for x uniform in the box: E f^2 - (E f)^2,
    E f^2 = 1/2 - 1/2 Re prod_d (e^{2 i b} - e^{2 i a}) / (2 i (b-a))."""
    mp.mp.dps = 40
    vol = mp.mpf(1)
    z1 = mp.mpc(1)
    z2 = mp.mpc(1)
    for a, b in zip(lower, upper):
        vol *= (b - a)
        z1 *= (mp.expj(b) - mp.expj(a)) / (mp.mpc(0, 1) * (b - a))
        z2 *= (mp.expj(2 * b) - mp.expj(2 * a)) / (mp.mpc(0, 2) * (b - a))
    ef = z1.imag
    ef2 = mp.mpf(0.5) - z2.real / 2
    return float(ef2 - ef * ef)


def ulp32(x) -> float:
    return float(np.spacing(np.float32(abs(x))))


# ---------------------------------------------------------------- GPU-vs-oracle comparison (parity rules P2-P4)
def compare_tree(it, ores, w: W.Workload, *, tol_sum=1e-12, tol_stat=1e-11, exact_sets=True):
    """Compare every level of a finished CUDA run `it` (binding.Integrator, keep_level_stats on) with
    the oracle result `ores` (oracle.run(..., keep_cells=True)) cell by cell.

    P2  per-(cell,trial) sums: |S_gpu - S_orc| <= tol_sum * N (|f| <= 1 for the bounded built-ins;
        callers with unbounded f pass a scaled tol_sum) -- only the FP64 summation order differs.
    P3  refined sets identical (exact mode).
    P4  value/std: relative 1e-6 is BASELINE.json's bar; tol_stat is what exact mode achieves.
    Returns the number of cells compared."""
    st = it.stats()
    n_cmp = 0
    assert st.overflow == 0
    for lev, ol in enumerate(ores.levels, start=1):
        gl = it.level_cells(lev)
        assert len(gl.mu) == ol.n_cells, (lev, len(gl.mu), ol.n_cells)
        assert st.level[lev - 1].n_cells == ol.n_cells
        assert st.level[lev - 1].n_refined == ol.n_refined
        np.testing.assert_array_equal(gl.instance, ol.instance)
        assert gl.path == ol.path
        scale = float(w.n_samples)
        dS = np.abs(gl.S - ol.S)
        assert dS.max() <= tol_sum * scale, (lev, dS.max())
        sc = max(np.abs(ol.mu).max(), ol.s.max(), 1e-300)
        assert np.abs(gl.mu - ol.mu).max() <= tol_stat * sc
        assert np.abs(gl.s - ol.s).max() <= 100 * tol_stat * sc
        # tau = mean(s) + m*pstd(s) is (1 + |m|)-Lipschitz in max|ds|: where s itself is ill-conditioned (cells so small that
        # f is constant to 9 digits) the thresholds inherit exactly that much and no more
        ds = float(np.abs(gl.s - ol.s).max())
        assert np.abs(gl.tau - ol.tau).max() <= 100 * tol_stat * max(np.abs(ol.tau).max(), 1e-300) + (1.0 + abs(w.sigma_multiplier)) * ds      # |tau|: m < 0 makes tau negative
        if exact_sets:
            np.testing.assert_array_equal(gl.refined, ol.refined)
        n_cmp += ol.n_cells
    for lev in range(len(ores.levels) + 1, w.depth + 1):   # levels the tree never reached
        assert st.level[lev - 1].n_cells == 0
    v, s = it.result()
    assert np.all(np.abs(v - ores.value) <= 1e-6 * np.maximum(np.abs(ores.value), 1e-300))
    assert np.all(np.abs(v - ores.value) <= tol_stat * np.maximum(np.abs(ores.value), ores.std))
    assert np.all(np.abs(s - ores.std) <= 1e-9 * np.maximum(ores.std, 1e-300))
    return n_cmp


def host_control(mu, s, k, level, depth, m, instance, budget=0, largest_spread=False):
    """Re-derive the control path (H7-H10) of one level in numpy from dumped per-cell (mu, s):
    per-group tau = mean + m*pstd (R6), flags s > tau for level < depth (R7), first-B budget per
    instance in path order (R12) or largest-spread-first (R14), accepted sums. Test-side restatement; shares nothing with either
    implementation. Returns (tau_per_cell, refined, acc_value[instance], acc_var[instance])."""
    n = len(mu)
    G = n // k
    sg = s.reshape(G, k)
    mean = sg.mean(axis=1)
    pstd = np.sqrt(((sg - mean[:, None]) ** 2).mean(axis=1))
    tau = mean + m * pstd
    tau_c = np.repeat(tau, k)
    flag = (s > tau_c) & (level < depth)
    refined = flag.copy()
    if budget > 0:
        for b in np.unique(instance):
            idx = np.nonzero(flag & (instance == b))[0]
            if largest_spread:      # R14: the B largest spreads, equal ones in path order
                idx = np.array(sorted(idx, key=lambda i: (-s[i], i)), dtype=np.int64)
            refined[idx[budget:]] = False
    ninst = int(instance.max()) + 1
    val = np.zeros(ninst)
    var = np.zeros(ninst)
    acc = ~refined
    np.add.at(val, instance[acc], mu[acc])
    np.add.at(var, instance[acc], s[acc] ** 2)
    return tau_c, refined, val, var
