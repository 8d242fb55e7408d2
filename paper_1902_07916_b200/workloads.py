"""Seeded synthetic workloads: the five BASELINE.json configs as plain data.

This module holds NO arithmetic of the method (no RNG stream, no map, no integrand, no
statistics). It only states problem sizes and generates the input parameter arrays, so it can
serve the oracle (tests) and the CUDA path alike ("Input recipe").

The paper measures on analytic integrands (Eq. 1 and 2), not on a dataset;
configs 2, 3 and 5 are those two integrands at BASELINE.json's sizes, configs 1 and 4 are
BASELINE.json's own.
"""
from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

# integrand / precision names shared by the binding and by tests (ids are resolved by each side)
CONST, LINEAR, SIN_SUM, EXP_QUAD = "const", "linear", "sin_sum", "exp_quad"
F64, F32 = "f64", "f32"


@dataclass(frozen=True)
class Workload:
    name: str
    dim: int
    lower: tuple
    upper: tuple
    g: int                      # divisions per axis
    n_samples: int              # N per cell per trial
    trials: int                 # T
    depth: int                  # L
    sigma_multiplier: float     # m
    seed: int
    integrand: str
    precision: str
    params: Optional[np.ndarray] = None   # [n_instances, params_per_instance], float64
    n_instances: int = 1
    max_groups_per_level: int = 0         # R12 refinement budget (0 = off = paper semantics)
    max_cells_per_level: int = 0          # capacity hint for one level (0 = library default); exceeding it is an error
    note: str = ""

    @property
    def k(self) -> int:
        return self.g ** self.dim

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


def gaussian_params(dim: int, sigma: float, centre: float = 0.0) -> np.ndarray:
    """EXP_QUAD parameters [A, a, c_0..c_{D-1}] of the paper's f2 (Eq. 2):
    A = (2 pi sigma^2)^(-D/2), a = 1/(2 sigma^2)."""
    A = (2.0 * np.pi * sigma * sigma) ** (-0.5 * dim)
    a = 1.0 / (2.0 * sigma * sigma)
    return np.array([[A, a] + [centre] * dim], dtype=np.float64)


def batched_params(n: int = 1024, dim: int = 4, seed: int = 4) -> np.ndarray:
    """Config 4 inputs: a_k log-uniform in [1, 1000], c_k uniform in [0.2, 0.8]^dim, seeded.
    Values are rounded to float32-representable numbers (the FP32 path would round them anyway;
    this keeps the closed form and the evaluated function the same function)."""
    rng = np.random.default_rng(seed)
    a = 10.0 ** (3.0 * rng.random(n))
    c = 0.2 + 0.6 * rng.random((n, dim))
    p = np.empty((n, 2 + dim), dtype=np.float64)
    p[:, 0] = 1.0
    p[:, 1] = a.astype(np.float32).astype(np.float64)
    p[:, 2:] = c.astype(np.float32).astype(np.float64)
    return p


def config1() -> Workload:
    return Workload("cfg1_sin3d_f64", 3, (0.0,) * 3, (10.0,) * 3, 4, 2000, 5, 2, 1.5, 1, SIN_SUM, F64,
                    note="BASELINE.json configs[0] (PR1 ref)")


def config2(depth: int = 3, budget: int = 0) -> Workload:
    return Workload("cfg2_sin6d", 6, (0.0,) * 6, (10.0,) * 6, 4, 100000, 5, depth, 1.5, 2, SIN_SUM, F32,
                    max_groups_per_level=budget, note="BASELINE.json configs[1]; paper f1, Eq. (1)")


def config3() -> Workload:
    return Workload("cfg3_gauss9d", 9, (-1.0,) * 9, (1.0,) * 9, 3, 20000, 5, 4, 1.0, 3, EXP_QUAD, F32,
                    params=gaussian_params(9, 0.01), max_cells_per_level=4 * 3 ** 9,
                    note="BASELINE.json configs[2]; paper f2, Eq. (2)")


def config4(n_instances: int = 1024) -> Workload:
    p = batched_params(1024, 4, 4)[:n_instances]
    return Workload("cfg4_batched4d", 4, (0.0,) * 4, (1.0,) * 4, 6, 4096, 5, 2, 1.5, 4, EXP_QUAD, F32,
                    params=p, n_instances=n_instances,
                    note="BASELINE.json configs[3]; sigma_multiplier unspecified there -> 1.5 (reading R11)")


def config5(depth: int = 4, budget: int = 0) -> Workload:
    return Workload("cfg5_sin6d_stress", 6, (0.0,) * 6, (10.0,) * 6, 8, 200000, 10, depth, 1.0, 5, SIN_SUM, F32,
                    max_groups_per_level=budget, note="BASELINE.json configs[4]")


def gauss12d() -> Workload:
    """the 12-D Gaussian of the paper's Table 4 at the paper's own sizes:
    3 divisions per axis (531441 cells), 1e4 samples per cell, 5 trials, depth 4, "4 sigma" threshold."""
    return Workload("cfg12_gauss12d", 12, (-1.0,) * 12, (1.0,) * 12, 3, 10000, 5, 4, 4.0, 12, EXP_QUAD, F32,
                    params=gaussian_params(12, 0.01), max_cells_per_level=4 * 3 ** 12,
                    note="paper Table 4 (PAPER.md:202-216); f2, Eq. (2), D = 12")


def paper_table3_sin6d() -> Workload:
    """The paper's Table 3 run of f1: 12 divisions per axis (2 985 984 cells), 1e4 samples per cell,
    5 trials, depth 1 -- 1.49e11 evaluations; 38.7 s on one V100, 298.8 s on one K40m."""
    return Workload("paper_t3_sin6d", 6, (0.0,) * 6, (10.0,) * 6, 12, 10000, 5, 1, 5.0, 33, SIN_SUM, F32,
                    note="paper Table 3 (PAPER.md:162-184); f1, Eq. (1)")


def paper_table4_gauss9d() -> Workload:
    """The paper's Table 4 run of f2 in 9-D: 3 divisions per axis, 1e4 samples per cell, 5 trials,
    depth 4, "4 sigma"; 4.8 s on one V100."""
    return Workload("paper_t4_gauss9d", 9, (-1.0,) * 9, (1.0,) * 9, 3, 10000, 5, 4, 4.0, 34, EXP_QUAD, F32,
                    params=gaussian_params(9, 0.01), max_cells_per_level=4 * 3 ** 9,
                    note="paper Table 4 (PAPER.md:202-216); f2, Eq. (2), D = 9")


# ---------------------------------------------------------------- vector-valued user integrands (R15)
# Inputs, not arithmetic of the method: CUDA device-function text handed to zmc_set_integrand_source_vec (and, `__device__`
# defined away, to g++ for the oracle). f_j(x) = (p0 * sum_d x_d)^(j+1), j = 0 .. n_out-1: n_out "terms" that share one sample
# stream -- the shape of the paper's application, an integrand of "several thousands terms".
VEC_MOMENTS_FN = "moments8"
VEC_MOMENTS_SRC = """
template <class R> __device__ inline void moments8_t(const R* x, int dim, const R* p, int np, R* out, int n_out) {
    R s = x[0];
    for (int d = 1; d < dim; ++d) s = s + x[d];
    R c = p[0] * s;
    R v = c;
    for (int j = 0; j < n_out; ++j) { out[j] = v; v = v * c; }
}
__device__ void moments8(const float* x, int dim, const float* p, int np, float* out, int n_out) { moments8_t<float>(x, dim, p, np, out, n_out); }
__device__ void moments8(const double* x, int dim, const double* p, int np, double* out, int n_out) { moments8_t<double>(x, dim, p, np, out, n_out); }
"""


def vec_moments6d(n_components: int = 8) -> Workload:
    """6-D, 4096 cells, 1e5 samples per cell, 5 trials, one level: BASELINE.json configs[1]'s sizes with the vector-valued integrand above
    (integrand/params are placeholders here: the function is VEC_MOMENTS_SRC, its parameter p0 = 0.3)."""
    return Workload("vec_moments6d_c%d" % n_components, 6, (0.0,) * 6, (1.0,) * 6, 4, 100000, 5, 1, 1.5, 6, CONST, F32,
                    params=np.array([[0.3]]), note="DESIGN.md R15: %d components, one sample stream" % n_components)
