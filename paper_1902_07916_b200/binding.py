"""Thin ctypes binding of libzmc.so (include/zmc.h). Argument marshalling only: every step of the
hot path -- Philox, map, integrand, reduction, statistics, threshold, flag, compaction, result --
runs in the CUDA kernels behind the C ABI. PyTorch supplies the stream and (optionally) the
workspace memory; nothing else.

There is no CPU fallback: if libzmc.so cannot be loaded or built, importing a symbol from it
raises, and without a CUDA device zmc_create fails with ZMC_ERR_CUDA.
"""
import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

from . import workloads as W

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libzmc.so")

# include/zmc.h
OK, ERR_ARG, ERR_RANGE, ERR_NO_INTEGRAND, ERR_COMPILE, ERR_CUDA, ERR_CAPACITY, ERR_NOT_RUN, ERR_STATE = 0, -1, -2, -3, -4, -5, -6, -7, -8
CONST, LINEAR, SIN_SUM, EXP_QUAD, USER = 0, 1, 2, 3, 100
OPT_PRECISION, OPT_MATH, OPT_MAX_GROUPS_PER_LEVEL, OPT_KEEP_LEVEL_STATS = 1, 2, 3, 4
OPT_MAX_CELLS_PER_LEVEL, OPT_GRID_BLOCKS, OPT_TARGET_ITEMS, OPT_USE_GRAPH = 5, 6, 7, 8
OPT_SPREAD, OPT_BUDGET_ORDER, OPT_SINGLE_LAUNCH = 9, 10, 11
SPREAD_TRIALS, SPREAD_SAMPLES = 0, 1
BUDGET_PATH_ORDER, BUDGET_LARGEST_SPREAD = 0, 1
F64, F32 = 0, 1
MATH_EXACT, MATH_FAST = 0, 1
MAX_DEPTH = 15

EXPORTS = ["zmc_create", "zmc_set_integrand", "zmc_set_integrand_source", "zmc_set_integrand_source_vec", "zmc_set_option", "zmc_workspace_bytes",
           "zmc_set_workspace", "zmc_run", "zmc_result", "zmc_stats", "zmc_level_cells", "zmc_level_cells_range", "zmc_level_sumsq", "zmc_debug_words",
           "zmc_debug_points", "zmc_flat_static", "zmc_last_error", "zmc_status_string", "zmc_destroy"]
STATIC_SCRATCH_BYTES, STATIC_MAX_CELLS, STATIC_MAX_UNITS, STATIC_MAX_PARAMS = 2 << 20, 4096, 131072, 32

_INTEGRAND_ID = {W.CONST: CONST, W.LINEAR: LINEAR, W.SIN_SUM: SIN_SUM, W.EXP_QUAD: EXP_QUAD}
_PRECISION_ID = {W.F64: F64, W.F32: F32}


class LevelStats(C.Structure):
    _fields_ = [("n_groups", C.c_uint64), ("n_cells", C.c_uint64), ("n_flagged", C.c_uint64),
                ("n_refined", C.c_uint64), ("evals", C.c_uint64), ("sample_ms", C.c_float), ("control_ms", C.c_float)]


class Stats(C.Structure):
    _fields_ = [("levels", C.c_int32), ("overflow", C.c_int32), ("nonfinite", C.c_uint64),
                ("total_evals", C.c_uint64), ("total_ms", C.c_float), ("regs_per_thread", C.c_int32),
                ("grid_blocks", C.c_int32), ("block_threads", C.c_int32), ("kernel_origin", C.c_int32),
                ("kernel_launches", C.c_int32), ("level", LevelStats * MAX_DEPTH)]


class ZmcError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("zmc status %d: %s" % (status, msg))
        self.status = status


_lib = None


def lib():
    """Load libzmc.so (building it first if nvcc is present and the sources changed)."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    if os.path.exists(_build.NVCC):
        path = _build.build()        # rebuilds iff the sources changed; a compile or link error is raised, never papered over
    elif os.path.exists(LIB_PATH):
        path = LIB_PATH              # no compiler on this machine: the shipped library as it is
        if not _build.is_current() and os.environ.get("ZMC_ALLOW_STALE") != "1":
            raise RuntimeError("libzmc.so does not match the sources (stamp mismatch) and there is no nvcc to rebuild it; "
                               "set ZMC_ALLOW_STALE=1 to load it anyway")
    else:
        raise RuntimeError("libzmc.so is missing and nvcc (%s) is not available to build it" % _build.NVCC)
    L = C.CDLL(path)
    vp, dp, u32p, u64p = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    L.zmc_create.argtypes = [C.POINTER(vp), C.c_int, dp, dp, C.c_int, C.c_uint64, C.c_int, C.c_int, C.c_double, C.c_uint64]
    L.zmc_set_integrand.argtypes = [vp, C.c_int, dp, C.c_int, C.c_int]
    L.zmc_set_integrand_source.argtypes = [vp, C.c_char_p, C.c_char_p, dp, C.c_int, C.c_int]
    L.zmc_set_integrand_source_vec.argtypes = [vp, C.c_char_p, C.c_char_p, C.c_int, dp, C.c_int, C.c_int]
    L.zmc_set_option.argtypes = [vp, C.c_int, C.c_int64]
    L.zmc_workspace_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    L.zmc_set_workspace.argtypes = [vp, vp, C.c_size_t]
    L.zmc_run.argtypes = [vp, vp]
    L.zmc_result.argtypes = [vp, dp, dp]
    L.zmc_stats.argtypes = [vp, C.POINTER(Stats)]
    L.zmc_level_cells.argtypes = [vp, C.c_int, C.c_uint64, u64p, u32p, u64p, u32p, dp, dp, dp, C.POINTER(C.c_uint8), dp]
    L.zmc_level_cells_range.argtypes = [vp, C.c_int, C.c_uint64, C.c_uint64, u32p, u64p, u32p, dp, dp, dp, C.POINTER(C.c_uint8), dp]
    L.zmc_level_sumsq.argtypes = [vp, C.c_int, C.c_uint64, dp]
    L.zmc_debug_words.argtypes = [vp, C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_uint64, C.c_uint64, u32p]
    L.zmc_debug_points.argtypes = [vp, C.c_uint32, C.c_uint64, C.c_uint32, C.c_int, u32p, C.c_int, C.c_uint64, dp, dp]
    L.zmc_flat_static.argtypes = [C.c_int, dp, dp, C.c_int, C.c_uint64, C.c_int, C.c_uint64, C.c_int, dp, C.c_int, C.c_int, C.c_int,
                                  vp, vp, C.c_char_p, C.c_size_t]
    L.zmc_last_error.argtypes = [vp]
    L.zmc_last_error.restype = C.c_char_p
    L.zmc_status_string.argtypes = [C.c_int]
    L.zmc_status_string.restype = C.c_char_p
    L.zmc_destroy.argtypes = [vp]
    L.zmc_destroy.restype = None
    _lib = L
    return L


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _ptr(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


@dataclass
class LevelCells:
    instance: np.ndarray
    path: list
    mu: np.ndarray
    s: np.ndarray
    tau: np.ndarray
    refined: np.ndarray
    S: np.ndarray


class Integrator:
    """One zmc_ctx. Methods carry the C names without the prefix."""

    def __init__(self, dim: int, lower: Sequence[float], upper: Sequence[float], divisions_per_axis: int,
                 samples_per_cell: int, trials: int, depth: int, sigma_multiplier: float, seed: int):
        self._L = lib()
        self._h = C.c_void_p()
        self.dim, self.trials, self.depth = dim, trials, depth
        self.n_instances = 1
        self.n_components = 0       # 0: scalar integrand; C >= 1: vector-valued user integrand, results carry a component axis
        lo = np.ascontiguousarray(lower, dtype=np.float64)
        up = np.ascontiguousarray(upper, dtype=np.float64)
        rc = self._L.zmc_create(C.byref(self._h), dim, _dp(lo), _dp(up), divisions_per_axis, samples_per_cell,
                                trials, depth, float(sigma_multiplier), seed)
        if rc != OK:      # no context exists after a failed zmc_create; the reason is zmc_last_error(NULL)
            raise ZmcError(rc, self._L.zmc_last_error(None).decode() or self._L.zmc_status_string(rc).decode())
        self._ws = None

    def _check(self, rc):
        if rc != OK:
            raise ZmcError(rc, self._L.zmc_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.zmc_destroy(self._h)
            self._h = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_integrand(self, builtin_id: int, params: Optional[np.ndarray] = None, n_instances: int = 1):
        if params is None:
            p, ppi = None, 0
        else:
            p = np.ascontiguousarray(params, dtype=np.float64).reshape(n_instances, -1)
            ppi = p.shape[1]
        self._check(self._L.zmc_set_integrand(self._h, builtin_id, _dp(p), ppi, n_instances))
        self.n_instances = n_instances
        self.n_components = 0

    def set_integrand_source(self, cuda_src: str, fn_name: str, params: Optional[np.ndarray] = None, n_instances: int = 1):
        if params is None:
            p, ppi = None, 0
        else:
            p = np.ascontiguousarray(params, dtype=np.float64).reshape(n_instances, -1)
            ppi = p.shape[1]
        self._check(self._L.zmc_set_integrand_source(self._h, cuda_src.encode(), fn_name.encode(), _dp(p), ppi, n_instances))
        self.n_instances = n_instances
        self.n_components = 0

    def set_integrand_source_vec(self, cuda_src: str, fn_name: str, n_components: int, params: Optional[np.ndarray] = None,
                                 n_instances: int = 1):
        if params is None:
            p, ppi = None, 0
        else:
            p = np.ascontiguousarray(params, dtype=np.float64).reshape(n_instances, -1)
            ppi = p.shape[1]
        self._check(self._L.zmc_set_integrand_source_vec(self._h, cuda_src.encode(), fn_name.encode(), n_components, _dp(p), ppi, n_instances))
        self.n_instances = n_instances
        self.n_components = n_components

    def _cshape(self, *lead):
        """Array shape of a per-`lead` quantity: a trailing component axis for vector-valued integrands."""
        return tuple(lead) + ((self.n_components,) if self.n_components else ())

    def set_option(self, key: int, value: int):
        self._check(self._L.zmc_set_option(self._h, key, int(value)))

    def workspace_bytes(self) -> int:
        n = C.c_size_t()
        self._check(self._L.zmc_workspace_bytes(self._h, C.byref(n)))
        return n.value

    def set_workspace(self, device_ptr: int, nbytes: int):
        self._check(self._L.zmc_set_workspace(self._h, C.c_void_p(device_ptr), nbytes))

    def use_torch_workspace(self):
        """Allocate the workspace as a torch uint8 tensor on the current CUDA device (kept alive here)."""
        import torch
        n = self.workspace_bytes()
        self._ws = torch.empty(n + 256, dtype=torch.uint8, device="cuda")
        p = (self._ws.data_ptr() + 255) & ~255
        self.set_workspace(p, n)

    def run(self, stream: Optional[int] = None):
        """Enqueue the whole tree search on `stream` (a raw cudaStream_t; default: torch's current stream)."""
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        self._check(self._L.zmc_run(self._h, C.c_void_p(stream)))

    def result(self):
        v = np.zeros(self._cshape(self.n_instances))
        s = np.zeros(self._cshape(self.n_instances))
        self._check(self._L.zmc_result(self._h, _dp(v), _dp(s)))
        return v, s

    def stats(self) -> Stats:
        st = Stats()
        self._check(self._L.zmc_stats(self._h, C.byref(st)))
        return st

    def level_cells(self, level: int) -> LevelCells:
        n = C.c_uint64()
        self._check(self._L.zmc_level_cells(self._h, level, 0, C.byref(n), None, None, None, None, None, None, None, None))
        n = n.value
        inst = np.zeros(n, dtype=np.uint32)
        plo = np.zeros(n, dtype=np.uint64)
        phi = np.zeros(n, dtype=np.uint32)
        mu, s, tau = np.zeros(self._cshape(n)), np.zeros(self._cshape(n)), np.zeros(self._cshape(n))
        ref = np.zeros(n, dtype=np.uint8)
        S = np.zeros(self._cshape(n, self.trials))
        nn = C.c_uint64()
        self._check(self._L.zmc_level_cells(self._h, level, n, C.byref(nn), _ptr(inst, C.c_uint32), _ptr(plo, C.c_uint64),
                                            _ptr(phi, C.c_uint32), _dp(mu), _dp(s), _dp(tau), _ptr(ref, C.c_uint8), _dp(S)))
        path = [(int(h) << 64) | int(l) for h, l in zip(phi, plo)]
        return LevelCells(inst, path, mu, s, tau, ref, S)

    def level_cells_range(self, level: int, first: int, count: int) -> LevelCells:
        inst = np.zeros(count, dtype=np.uint32)
        plo = np.zeros(count, dtype=np.uint64)
        phi = np.zeros(count, dtype=np.uint32)
        mu, s, tau = np.zeros(self._cshape(count)), np.zeros(self._cshape(count)), np.zeros(self._cshape(count))
        ref = np.zeros(count, dtype=np.uint8)
        S = np.zeros(self._cshape(count, self.trials))
        self._check(self._L.zmc_level_cells_range(self._h, level, first, count, _ptr(inst, C.c_uint32), _ptr(plo, C.c_uint64),
                                                  _ptr(phi, C.c_uint32), _dp(mu), _dp(s), _dp(tau), _ptr(ref, C.c_uint8), _dp(S)))
        path = [(int(h) << 64) | int(l) for h, l in zip(phi, plo)]
        return LevelCells(inst, path, mu, s, tau, ref, S)

    def level_stats_range(self, level: int, first: int, count: int):
        """(mu, s, refined) of the cells [first, first + count) of one level, without identities and per-trial sums: what a pass over a
        level of 10^8 cells needs (zmc_level_cells_range with the other arrays NULL)."""
        mu, s = np.zeros(self._cshape(count)), np.zeros(self._cshape(count))
        ref = np.zeros(count, dtype=np.uint8)
        self._check(self._L.zmc_level_cells_range(self._h, level, first, count, None, None, None, _dp(mu), _dp(s), None,
                                                  _ptr(ref, C.c_uint8), None))
        return mu, s, ref

    def level_sumsq(self, level: int, n_cells: int) -> np.ndarray:
        Q = np.zeros(self._cshape(n_cells, self.trials))
        self._check(self._L.zmc_level_sumsq(self._h, level, n_cells, _dp(Q)))
        return Q

    def debug_words(self, instance: int, path: int, level: int, trial: int, first_word: int, n_words: int) -> np.ndarray:
        out = np.zeros(n_words, dtype=np.uint32)
        self._check(self._L.zmc_debug_words(self._h, instance, path & (2 ** 64 - 1), path >> 64, level, trial,
                                            first_word, n_words, _ptr(out, C.c_uint32)))
        return out

    def debug_points(self, instance: int, path: int, level: int, coords, trial: int, n: int):
        cc = np.ascontiguousarray(coords, dtype=np.uint32)
        x = np.zeros((n, self.dim))
        f = np.zeros(self._cshape(n))
        self._check(self._L.zmc_debug_points(self._h, instance, path & (2 ** 64 - 1), path >> 64, level,
                                             _ptr(cc, C.c_uint32), trial, n, _dp(x), _dp(f)))
        return x, f


def flat_static(dim: int, lower: Sequence[float], upper: Sequence[float], divisions_per_axis: int, samples_per_cell: int, trials: int,
                seed: int, builtin_id: int, params: Optional[np.ndarray], precision: int, math: int, result_device_ptr: int,
                stream: Optional[int] = None) -> None:
    """zmc_flat_static: one level of stratified sampling whose scratch memory is a fixed array inside libzmc.so -- the call for hosts
    that cannot allocate device memory (the card is owned by somebody else's pool, or cudaMalloc's synchronisation is not acceptable).
    `result_device_ptr` is the address of 2 doubles in device memory that the caller owns (value, std); they are valid once `stream`
    has finished. Nothing is allocated and nothing is synchronised here; calls that overlap on the GPU share the scratch and race."""
    L = lib()
    lo = np.ascontiguousarray(lower, dtype=np.float64)
    up = np.ascontiguousarray(upper, dtype=np.float64)
    p = None if params is None else np.ascontiguousarray(params, dtype=np.float64).reshape(-1)
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    err = C.create_string_buffer(512)
    rc = L.zmc_flat_static(dim, _dp(lo), _dp(up), divisions_per_axis, samples_per_cell, trials, seed, builtin_id, _dp(p),
                           0 if p is None else p.size, precision, math, C.c_void_p(result_device_ptr), C.c_void_p(stream), err, len(err))
    if rc != OK:
        raise ZmcError(rc, err.value.decode())


def from_workload(w: W.Workload, math: int = MATH_EXACT, keep_level_stats: bool = False,
                  max_cells_per_level: int = 0, use_graph: bool = False, spread: int = SPREAD_TRIALS,
                  budget_order: int = BUDGET_PATH_ORDER, single_launch: Optional[int] = None) -> Integrator:
    """zmc_create + zmc_set_integrand + options for one of the seeded workloads."""
    it = Integrator(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.depth, w.sigma_multiplier, w.seed)
    it.set_integrand(_INTEGRAND_ID[w.integrand], w.params, w.n_instances)
    it.set_option(OPT_PRECISION, _PRECISION_ID[w.precision])
    it.set_option(OPT_MATH, math)
    if w.max_groups_per_level:
        it.set_option(OPT_MAX_GROUPS_PER_LEVEL, w.max_groups_per_level)
    if keep_level_stats:
        it.set_option(OPT_KEEP_LEVEL_STATS, 1)
    if use_graph:
        it.set_option(OPT_USE_GRAPH, 1)
    if single_launch is not None:
        it.set_option(OPT_SINGLE_LAUNCH, single_launch)
    if spread != SPREAD_TRIALS:
        it.set_option(OPT_SPREAD, spread)
    if budget_order != BUDGET_PATH_ORDER:
        it.set_option(OPT_BUDGET_ORDER, budget_order)
    if max_cells_per_level or w.max_cells_per_level:
        it.set_option(OPT_MAX_CELLS_PER_LEVEL, max_cells_per_level or w.max_cells_per_level)
    return it
