"""Test helpers: closed forms (independent of oracle/ and of the CUDA path) and
Workload -> oracle.Config conversion."""
import math

import mpmath as mp
import numpy as np

import oracle as O
from paper_1902_07916_b200 import workloads as W

_ORC_INTEGRAND = {W.CONST: O.CONST, W.LINEAR: O.LINEAR, W.SIN_SUM: O.SIN_SUM, W.EXP_QUAD: O.EXP_QUAD}
_ORC_PRECISION = {W.F64: O.F64, W.F32: O.F32}


def oracle_config(w: W.Workload, **over) -> O.Config:
    cfg = O.Config(dim=w.dim, lower=list(w.lower), upper=list(w.upper), g=w.g, n_samples=w.n_samples,
                   trials=w.trials, depth=w.depth, sigma_multiplier=w.sigma_multiplier, seed=w.seed,
                   integrand=_ORC_INTEGRAND[w.integrand], precision=_ORC_PRECISION[w.precision],
                   params=w.params, n_instances=w.n_instances, max_groups_per_level=w.max_groups_per_level)
    for k, v in over.items():
        setattr(cfg, k, v)
    return cfg


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
