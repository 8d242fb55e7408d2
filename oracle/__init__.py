"""ORACLE -- test infrastructure, NOT the product.

ctypes loader for oracle/libzmc_oracle.so (plain single-threaded C++; see
zmc_oracle.h). Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the product
(paper_1902_07916_b200) never does.
"""
import ctypes as C
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

from . import build as _build

CONST, LINEAR, SIN_SUM, EXP_QUAD = 0, 1, 2, 3
F64, F32 = 0, 1
SCOPE_GROUP, SCOPE_POOLED = 0, 1
BFS, DFS = 0, 1
SPREAD_TRIALS, SPREAD_SAMPLES = 0, 1              # R13
BUDGET_PATH_ORDER, BUDGET_LARGEST_SPREAD = 0, 1   # R14


class _Cfg(C.Structure):
    _fields_ = [
        ("dim", C.c_int32), ("g", C.c_int32), ("trials", C.c_int32), ("depth", C.c_int32),
        ("n_samples", C.c_uint64), ("seed", C.c_uint64), ("sigma_multiplier", C.c_double),
        ("integrand", C.c_int32), ("precision", C.c_int32), ("n_instances", C.c_int32),
        ("params_per_instance", C.c_int32), ("threshold_scope", C.c_int32), ("traversal", C.c_int32),
        ("max_groups_per_level", C.c_int64), ("spread", C.c_int32), ("budget_order", C.c_int32),
        ("lower", C.POINTER(C.c_double)), ("upper", C.POINTER(C.c_double)), ("params", C.POINTER(C.c_double)),
    ]


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(_build.build())
    u32p, u64p, dp = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_double)
    L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
    L.orc_derive_key.argtypes = [C.c_uint64, C.c_uint32, u32p]
    L.orc_unit_words.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_uint64, C.c_uint64, u32p]
    L.orc_cell_geometry.argtypes = [C.c_int, dp, dp, C.c_int, C.c_int, u32p, dp, dp, dp]
    L.orc_map_f64.argtypes = [C.c_uint32, C.c_double, C.c_double]
    L.orc_map_f64.restype = C.c_double
    L.orc_map_f32.argtypes = [C.c_uint32, C.c_double, C.c_double, C.c_double]
    L.orc_map_f32.restype = C.c_float
    L.orc_zsin.argtypes = [C.c_float]
    L.orc_zsin.restype = C.c_float
    L.orc_zexp.argtypes = [C.c_float, C.POINTER(C.c_int32)]
    L.orc_zexp.restype = C.c_float
    L.orc_zexp_value.argtypes = [C.c_float]
    L.orc_zexp_value.restype = C.c_double
    L.orc_unit_sum.argtypes = [C.POINTER(_Cfg), C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, u32p, C.c_int, dp, dp]
    L.orc_unit_sums.argtypes = [C.POINTER(_Cfg), C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, u32p, C.c_int, dp, dp]
    L.orc_cell_stats_samples.argtypes = [dp, dp, C.c_int, C.c_double, C.c_double, C.c_uint64, dp, dp]
    L.orc_level_sumsq.argtypes = [C.c_void_p, C.c_int, dp]
    L.orc_level_sumsq.restype = C.c_int64
    L.orc_unit_points.argtypes = [C.POINTER(_Cfg), C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, u32p, C.c_int, C.c_uint64, dp, dp]
    L.orc_cell_stats.argtypes = [dp, C.c_int, C.c_double, C.c_double, C.c_uint64, dp, dp, dp]
    L.orc_threshold.argtypes = [dp, C.c_int64, C.c_double]
    L.orc_threshold.restype = C.c_double
    L.orc_run.argtypes = [C.POINTER(_Cfg), C.c_int]
    L.orc_run.restype = C.c_void_p
    L.orc_free.argtypes = [C.c_void_p]
    L.orc_error.argtypes = [C.c_void_p]
    L.orc_error.restype = C.c_char_p
    L.orc_get.argtypes = [C.c_void_p, dp, dp]
    L.orc_levels.argtypes = [C.c_void_p]
    L.orc_level_counts.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.orc_total_evals.argtypes = [C.c_void_p]
    L.orc_total_evals.restype = C.c_uint64
    L.orc_level_cells.argtypes = [C.c_void_p, C.c_int, u32p, u64p, u32p, dp, dp, dp, C.POINTER(C.c_uint8), dp]
    L.orc_level_cells.restype = C.c_int64
    _lib = L
    return L


def config_from_workload(w, **over) -> "Config":
    """A seeded workload description (any object with the fields of paper_1902_07916_b200.workloads.Workload: plain sizes,
    names and parameter arrays -- this package imports nothing from the product) as an oracle Config."""
    integrand = {"const": CONST, "linear": LINEAR, "sin_sum": SIN_SUM, "exp_quad": EXP_QUAD}[w.integrand]
    precision = {"f64": F64, "f32": F32}[w.precision]
    cfg = Config(dim=w.dim, lower=list(w.lower), upper=list(w.upper), g=w.g, n_samples=w.n_samples,
                 trials=w.trials, depth=w.depth, sigma_multiplier=w.sigma_multiplier, seed=w.seed,
                 integrand=integrand, precision=precision, params=w.params, n_instances=w.n_instances,
                 max_groups_per_level=w.max_groups_per_level)
    for k, v in over.items():
        setattr(cfg, k, v)
    return cfg


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _u32p(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint32))


@dataclass
class Config:
    """One integration problem (mirrors orc_config)."""
    dim: int
    lower: Sequence[float]
    upper: Sequence[float]
    g: int
    n_samples: int
    trials: int
    depth: int
    sigma_multiplier: float
    seed: int
    integrand: int
    precision: int = F64
    params: Optional[np.ndarray] = None      # [n_instances, params_per_instance]
    n_instances: int = 1
    threshold_scope: int = SCOPE_GROUP
    traversal: int = BFS
    max_groups_per_level: int = 0
    spread: int = SPREAD_TRIALS
    budget_order: int = BUDGET_PATH_ORDER
    _keep: list = field(default_factory=list, repr=False)

    def c(self) -> _Cfg:
        lo = np.ascontiguousarray(self.lower, dtype=np.float64)
        up = np.ascontiguousarray(self.upper, dtype=np.float64)
        if self.params is None:
            p = np.zeros((self.n_instances, 1), dtype=np.float64)
            ppi = 0
        else:
            p = np.ascontiguousarray(self.params, dtype=np.float64).reshape(self.n_instances, -1)
            ppi = p.shape[1]
        self._keep[:] = [lo, up, p]
        return _Cfg(self.dim, self.g, self.trials, self.depth, self.n_samples, self.seed, self.sigma_multiplier,
                    self.integrand, self.precision, self.n_instances, ppi, self.threshold_scope, self.traversal,
                    self.max_groups_per_level, self.spread, self.budget_order, _dp(lo), _dp(up), _dp(p))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_u32p(c), _u32p(k), _u32p(out))
    return out


def derive_key(seed, instance=0):
    out = np.zeros(2, dtype=np.uint32)
    lib().orc_derive_key(seed, instance, _u32p(out))
    return out


def unit_words(seed, instance, path, level, trial, first_word, n_words):
    out = np.zeros(n_words, dtype=np.uint32)
    lib().orc_unit_words(seed, instance, path & (2**64 - 1), path >> 64, level, trial, first_word, n_words, _u32p(out))
    return out


def cell_geometry(dim, lower, upper, g, level, coords):
    lo_in = np.ascontiguousarray(lower, dtype=np.float64)
    up_in = np.ascontiguousarray(upper, dtype=np.float64)
    cc = np.ascontiguousarray(coords, dtype=np.uint32)
    lo = np.zeros(dim)
    w = np.zeros(dim)
    V = C.c_double()
    lib().orc_cell_geometry(dim, _dp(lo_in), _dp(up_in), g, level, _u32p(cc), _dp(lo), _dp(w), C.byref(V))
    return lo, w, V.value


def map_f64(w, lo, width):
    return lib().orc_map_f64(int(w), lo, width)


def map_f32(w, lo, width, centre=0.0):
    return np.float32(lib().orc_map_f32(int(w), lo, width, centre))


def zsin(a):
    return np.float32(lib().orc_zsin(float(np.float32(a))))


def zexp(e):
    n = C.c_int32()
    p = lib().orc_zexp(float(np.float32(e)), C.byref(n))
    return np.float32(p), n.value


def zexp_value(e):
    return lib().orc_zexp_value(float(np.float32(e)))


def path_coords(dim, g, path_digits):
    """Integer coordinates and path id of the cell reached by child indices `path_digits` (R2)."""
    k = g ** dim
    coords = [0] * dim
    P = 0
    for j in path_digits:
        P = P * k + j
        rem = j
        for d in range(dim):
            coords[d] = coords[d] * g + rem % g
            rem //= g
    return P, coords


def unit_sum(cfg: Config, instance, path, level, coords, trial):
    cc = np.ascontiguousarray(coords, dtype=np.uint32)
    S, Sabs = C.c_double(), C.c_double()
    c = cfg.c()
    rc = lib().orc_unit_sum(C.byref(c), instance, path & (2**64 - 1), path >> 64, level, _u32p(cc), trial,
                            C.byref(S), C.byref(Sabs))
    if rc != 0:
        raise ValueError("oracle: bad config")
    return S.value, Sabs.value


def unit_sums(cfg: Config, instance, path, level, coords, trial):
    """R13: (S, Q) = (sum f, sum f^2) of one unit."""
    cc = np.ascontiguousarray(coords, dtype=np.uint32)
    S, Q = C.c_double(), C.c_double()
    c = cfg.c()
    rc = lib().orc_unit_sums(C.byref(c), instance, path & (2**64 - 1), path >> 64, level, _u32p(cc), trial,
                             C.byref(S), C.byref(Q))
    if rc != 0:
        raise ValueError("oracle: bad config")
    return S.value, Q.value


def cell_stats_samples(S, Q, volume, prefactor, n_samples):
    S = np.ascontiguousarray(S, dtype=np.float64)
    Q = np.ascontiguousarray(Q, dtype=np.float64)
    mu, s = C.c_double(), C.c_double()
    lib().orc_cell_stats_samples(_dp(S), _dp(Q), len(S), volume, prefactor, n_samples, C.byref(mu), C.byref(s))
    return mu.value, s.value


def unit_points(cfg: Config, instance, path, level, coords, trial, n):
    cc = np.ascontiguousarray(coords, dtype=np.uint32)
    x = np.zeros((n, cfg.dim))
    f = np.zeros(n)
    c = cfg.c()
    rc = lib().orc_unit_points(C.byref(c), instance, path & (2**64 - 1), path >> 64, level, _u32p(cc), trial, n, _dp(x), _dp(f))
    if rc != 0:
        raise ValueError("oracle: bad config")
    return x, f


def cell_stats(S, volume, prefactor, n_samples):
    S = np.ascontiguousarray(S, dtype=np.float64)
    I = np.zeros_like(S)
    mu, s = C.c_double(), C.c_double()
    lib().orc_cell_stats(_dp(S), len(S), volume, prefactor, n_samples, _dp(I), C.byref(mu), C.byref(s))
    return I, mu.value, s.value


def threshold(s, m):
    s = np.ascontiguousarray(s, dtype=np.float64)
    return lib().orc_threshold(_dp(s), len(s), m)


@dataclass
class Level:
    n_cells: int
    n_refined: int
    n_truncated: int
    instance: Optional[np.ndarray] = None
    path: Optional[list] = None
    mu: Optional[np.ndarray] = None
    s: Optional[np.ndarray] = None
    tau: Optional[np.ndarray] = None
    refined: Optional[np.ndarray] = None
    S: Optional[np.ndarray] = None
    Q: Optional[np.ndarray] = None


@dataclass
class Result:
    value: np.ndarray
    std: np.ndarray
    levels: list
    evals: int


def run(cfg: Config, keep_cells: bool = False) -> Result:
    L = lib()
    c = cfg.c()
    h = L.orc_run(C.byref(c), 1 if keep_cells else 0)
    try:
        err = L.orc_error(h)
        if err:
            raise ValueError("oracle: " + err.decode())
        value = np.zeros(cfg.n_instances)
        std = np.zeros(cfg.n_instances)
        L.orc_get(h, _dp(value), _dp(std))
        levels = []
        for lev in range(1, L.orc_levels(h) + 1):
            a, b, t = C.c_int64(), C.c_int64(), C.c_int64()
            L.orc_level_counts(h, lev, C.byref(a), C.byref(b), C.byref(t))
            rec = Level(a.value, b.value, t.value)
            if keep_cells:
                n = a.value
                inst = np.zeros(n, dtype=np.uint32)
                plo = np.zeros(n, dtype=np.uint64)
                phi = np.zeros(n, dtype=np.uint32)
                mu, s, tau = np.zeros(n), np.zeros(n), np.zeros(n)
                ref = np.zeros(n, dtype=np.uint8)
                S = np.zeros((n, cfg.trials))
                L.orc_level_cells(h, lev, _u32p(inst), plo.ctypes.data_as(C.POINTER(C.c_uint64)), _u32p(phi),
                                  _dp(mu), _dp(s), _dp(tau), ref.ctypes.data_as(C.POINTER(C.c_uint8)), _dp(S))
                rec.instance, rec.mu, rec.s, rec.tau, rec.refined, rec.S = inst, mu, s, tau, ref, S
                rec.path = [int(phi[i]) << 64 | int(plo[i]) for i in range(n)]
                if cfg.spread == SPREAD_SAMPLES:
                    Q = np.zeros((n, cfg.trials))
                    L.orc_level_sumsq(h, lev, _dp(Q))
                    rec.Q = Q
            levels.append(rec)
        return Result(value, std, levels, L.orc_total_evals(h))
    finally:
        L.orc_free(h)


# ------------------------------------------------------------------ R15: vector-valued user integrands (zmc_oracle_vec.cpp)
USER_F64 = C.CFUNCTYPE(None, C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_double), C.c_int)
USER_F32 = C.CFUNCTYPE(None, C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_float), C.c_int)


def compile_user_fn(src: str, fn_name: str, precisions=("f64", "f32")):
    """Compile a user integrand -- the very text handed to zmc_set_integrand_source_vec, `__device__` defined away --
    with g++ (-O2 -ffp-contract=off, like the oracle) and return (f64, f32) C function pointers (None where not asked
    for). The user function is an input of the method, not part of it. The text must be plain C++ valid on both sides."""
    import hashlib
    import os
    import subprocess
    import tempfile
    wrap = ["#include <math.h>\n#define __device__\n#define __forceinline__ inline\n", src, "\n"]
    if "f64" in precisions:
        wrap.append('extern "C" void orc_user_entry_f64(const double* x, int dim, const double* p, int np, double* out, int n_out) '
                    "{ %s(x, dim, p, np, out, n_out); }\n" % fn_name)
    if "f32" in precisions:
        wrap.append('extern "C" void orc_user_entry_f32(const float* x, int dim, const float* p, int np, float* out, int n_out) '
                    "{ %s(x, dim, p, np, out, n_out); }\n" % fn_name)
    text = "".join(wrap)
    # a directory of this user's own (0700, ownership and mode checked): a library found there was put there by this user, and nobody else
    # can plant one under the predictable name; source and library are written under pid-unique names and renamed into place
    d = os.path.join(tempfile.gettempdir(), "zmc_oracle_user_%d" % os.getuid())
    os.makedirs(d, mode=0o700, exist_ok=True)
    st = os.lstat(d)
    import stat as _stat
    if not _stat.S_ISDIR(st.st_mode) or st.st_uid != os.getuid() or (st.st_mode & 0o077):
        raise RuntimeError("%s is not a directory owned by this user with mode 0700: refusing to load libraries from it" % d)
    tag = hashlib.sha256(text.encode()).hexdigest()[:24]
    so = os.path.join(d, "user_%s.so" % tag)
    if not os.path.exists(so):
        cpp = os.path.join(d, "user_%s.%d.cpp" % (tag, os.getpid()))
        with open(cpp, "w") as f:
            f.write(text)
        tmp = so + ".tmp%d" % os.getpid()
        try:
            subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-mfma", "-fPIC", "-shared", "-o", tmp, cpp], check=True)
            os.replace(tmp, so)
        finally:
            os.remove(cpp)
    L = C.CDLL(so)
    f64 = C.cast(L.orc_user_entry_f64, USER_F64) if "f64" in precisions else None
    f32 = C.cast(L.orc_user_entry_f32, USER_F32) if "f32" in precisions else None
    return f64, f32


def _vec_lib():
    L = lib()
    if not getattr(L, "_vec_ready", False):
        u32p, u64p, dp = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_double)
        L.orc_vec_unit_sums.argtypes = [C.POINTER(_Cfg), C.c_int, USER_F64, USER_F32, C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, u32p, C.c_int, dp]
        L.orc_run_vec.argtypes = [C.POINTER(_Cfg), C.c_int, USER_F64, USER_F32, C.c_int]
        L.orc_run_vec.restype = C.c_void_p
        L.orc_vec_free.argtypes = [C.c_void_p]
        L.orc_vec_error.argtypes = [C.c_void_p]
        L.orc_vec_error.restype = C.c_char_p
        L.orc_vec_get.argtypes = [C.c_void_p, dp, dp]
        L.orc_vec_levels.argtypes = [C.c_void_p]
        L.orc_vec_total_evals.argtypes = [C.c_void_p]
        L.orc_vec_total_evals.restype = C.c_uint64
        L.orc_vec_level_counts.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.orc_vec_level_cells.argtypes = [C.c_void_p, C.c_int, u32p, u64p, u32p, dp, dp, dp, C.POINTER(C.c_uint8), dp]
        L.orc_vec_level_cells.restype = C.c_int64
        L.orc_vec_level_sumsq.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_vec_level_sumsq.restype = C.c_int64
        L.orc_vec_unit_sums_sq.argtypes = [C.POINTER(_Cfg), C.c_int, USER_F64, USER_F32, C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, u32p, C.c_int, dp, dp]
        L._vec_ready = True
    return L


def _fn_args(fns):
    f64, f32 = fns
    return (f64 if f64 is not None else C.cast(None, USER_F64)), (f32 if f32 is not None else C.cast(None, USER_F32))


def vec_unit_sums(cfg: Config, n_components, fns, instance, path, level, coords, trial):
    """R15: the n_components sums of one (cell, trial) unit. fns = compile_user_fn(...)."""
    cc = np.ascontiguousarray(coords, dtype=np.uint32)
    S = np.zeros(n_components)
    c = cfg.c()
    f64, f32 = _fn_args(fns)
    rc = _vec_lib().orc_vec_unit_sums(C.byref(c), n_components, f64, f32, instance, path & (2**64 - 1), path >> 64, level,
                                      _u32p(cc), trial, _dp(S))
    if rc != 0:
        raise ValueError("oracle: bad config")
    return S


def vec_unit_sums_sq(cfg: Config, n_components, fns, instance, path, level, coords, trial):
    """R13 + R15: (S, Q), the n_components sums of f and of f^2 of one (cell, trial) unit."""
    cc = np.ascontiguousarray(coords, dtype=np.uint32)
    S, Q = np.zeros(n_components), np.zeros(n_components)
    c = cfg.c()
    f64, f32 = _fn_args(fns)
    rc = _vec_lib().orc_vec_unit_sums_sq(C.byref(c), n_components, f64, f32, instance, path & (2**64 - 1), path >> 64, level,
                                         _u32p(cc), trial, _dp(S), _dp(Q))
    if rc != 0:
        raise ValueError("oracle: bad config")
    return S, Q


def run_vec(cfg: Config, n_components, fns, keep_cells: bool = False) -> Result:
    """R15: the whole tree of a vector-valued user integrand. value, std: [n_instances, n_components];
    per level (keep_cells) mu, s, tau: [cells, C], S: [cells, T, C]."""
    L = _vec_lib()
    c = cfg.c()
    f64, f32 = _fn_args(fns)
    h = L.orc_run_vec(C.byref(c), n_components, f64, f32, 1 if keep_cells else 0)
    try:
        err = L.orc_vec_error(h)
        if err:
            raise ValueError("oracle: " + err.decode())
        nc = n_components
        value = np.zeros((cfg.n_instances, nc))
        std = np.zeros((cfg.n_instances, nc))
        L.orc_vec_get(h, _dp(value), _dp(std))
        levels = []
        for lev in range(1, L.orc_vec_levels(h) + 1):
            a, b, t = C.c_int64(), C.c_int64(), C.c_int64()
            L.orc_vec_level_counts(h, lev, C.byref(a), C.byref(b), C.byref(t))
            rec = Level(a.value, b.value, t.value)
            if keep_cells:
                n = a.value
                inst = np.zeros(n, dtype=np.uint32)
                plo = np.zeros(n, dtype=np.uint64)
                phi = np.zeros(n, dtype=np.uint32)
                mu, s, tau = np.zeros((n, nc)), np.zeros((n, nc)), np.zeros((n, nc))
                ref = np.zeros(n, dtype=np.uint8)
                S = np.zeros((n, cfg.trials, nc))
                L.orc_vec_level_cells(h, lev, _u32p(inst), plo.ctypes.data_as(C.POINTER(C.c_uint64)), _u32p(phi),
                                      _dp(mu), _dp(s), _dp(tau), ref.ctypes.data_as(C.POINTER(C.c_uint8)), _dp(S))
                rec.instance, rec.mu, rec.s, rec.tau, rec.refined, rec.S = inst, mu, s, tau, ref, S
                rec.path = [int(phi[i]) << 64 | int(plo[i]) for i in range(n)]
                if cfg.spread == SPREAD_SAMPLES:
                    Q = np.zeros((n, cfg.trials, nc))
                    L.orc_vec_level_sumsq(h, lev, _dp(Q))
                    rec.Q = Q
            levels.append(rec)
        return Result(value, std, levels, L.orc_vec_total_evals(h))
    finally:
        L.orc_vec_free(h)
