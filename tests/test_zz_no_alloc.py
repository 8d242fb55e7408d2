"""zmc_flat_static: the one entry point of libzmc.so that allocates no device memory.

Some hosts of this library cannot allocate on the GPU at all: a process in which another component's memory pool already holds the whole
card (any further cudaMalloc fails), or a latency-critical loop that must not run into the device-wide synchronisation that cudaMalloc
and cudaFree bring. zmc_run is no use to them (it allocates a workspace, or wants one that somebody allocated); zmc_flat_static keeps
all of its scratch in a fixed 2 MiB array inside the library image instead, which caps the problem size and is shared by every call.

This file is named so that pytest collects it LAST: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests. It depends on nothing the other tests leave behind: it passes alone in a fresh process and after the whole suite.

What is checked, against the existing path (zmc_create(depth = 1) + zmc_set_integrand + zmc_run + zmc_result):
  - the same value and std within the tolerances tests/helpers.compare_tree uses for results (1e-11 of max(|value|, std) on the value, 1e-9
    relative on the std) -- on two calls in a row, and again after a call with a different, smaller problem has left its contents in
    the shared array (a call must never depend on what the array held before);
  - the second call takes no device memory (cudaMemGetInfo's free bytes do not drop across it);
  - a problem beyond the fixed maximum is refused with an error that names the limit, and launches nothing.
"""
import numpy as np
import pytest

from paper_1902_07916_b200 import binding as B, workloads as W

pytestmark = pytest.mark.gpu

_ID = {W.CONST: B.CONST, W.LINEAR: B.LINEAR, W.SIN_SUM: B.SIN_SUM, W.EXP_QUAD: B.EXP_QUAD}
_PREC = {W.F64: B.F64, W.F32: B.F32}


def _flat(w: W.Workload) -> W.Workload:
    return w.with_(depth=1, max_groups_per_level=0, max_cells_per_level=0)


def _cases():
    """One-level problems inside the static limits (k <= 4096 cells, k * T <= 131072 units), one per code path of the sampling kernel:
    FP64 sin (chunked units), FP32 sin at the full 4096 cells, FP32 Gaussian (prefactor applied per trial, R8), a ragged sample tail."""
    gauss4 = W.Workload("gauss4d_f32", 4, (-1.0,) * 4, (1.0,) * 4, 6, 3001, 7, 1, 1.5, 11, W.EXP_QUAD, W.F32,
                        params=W.gaussian_params(4, 0.25, 0.125))
    lin5 = W.Workload("linear5d_f64", 5, (0.0, -1.0, 2.0, 0.5, -3.0), (1.0, 1.0, 2.5, 4.0, -1.0), 3, 777, 3, 1, 1.5, 12, W.LINEAR, W.F64,
                      params=np.array([[0.5, 1.0, -2.0, 3.0, 0.25, -0.75]]))
    return [_flat(W.config1()), _flat(W.config2()).with_(n_samples=20000), gauss4, lin5]


def _existing_path(w: W.Workload):
    """value, std of the one instance through zmc_create / zmc_set_integrand / zmc_run / zmc_result."""
    it = B.from_workload(w)
    try:
        it.run()
        v, s = it.result()
    finally:
        it.close()
    return float(v[0]), float(s[0])


def _static_path(w: W.Workload, out):
    """Enqueue zmc_flat_static on torch's current stream; `out` is the caller's 2-double device buffer."""
    B.flat_static(w.dim, w.lower, w.upper, w.g, w.n_samples, w.trials, w.seed, _ID[w.integrand], w.params, _PREC[w.precision],
                  B.MATH_EXACT, out.data_ptr())


def _agree(got, want, what):
    v, s = got
    v0, s0 = want
    assert np.isfinite(v) and np.isfinite(s), (what, got)
    assert abs(v - v0) <= 1e-11 * max(abs(v0), s0), (what, got, want)
    assert abs(s - s0) <= 1e-9 * max(s0, 1e-300), (what, got, want)


def test_flat_static_matches_the_existing_path_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available()
    cases = _cases()
    want = [_existing_path(w) for w in cases]
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")     # the caller's output; the entry point allocates nothing

    identical = 0
    for rounds in range(2):                     # every case twice in a row, then the next: each call finds the previous one's scratch
        for w, ref in zip(cases, want):
            for call in range(2):
                out.fill_(float("nan"))
                _static_path(w, out)
                got = tuple(out.cpu().tolist())  # synchronises the stream
                _agree(got, ref, "%s round %d call %d" % (w.name, rounds, call))
                identical += int(got == ref)
    # same device functions, same reduction shapes: in practice the results are the same bits; reported, the tolerance is the test
    print("zmc_flat_static: %d of %d results bit-identical to the existing path" % (identical, 4 * len(cases)))


def test_flat_static_takes_no_device_memory():
    import torch
    w = _cases()[1]
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    _static_path(w, out)                         # the first call on the device: address look-up, kernels loaded
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    _static_path(w, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)
    _agree(tuple(out.cpu().tolist()), _existing_path(w), w.name)


def test_flat_static_refuses_what_does_not_fit():
    import torch
    out = torch.full((2,), -7.0, dtype=torch.float64, device="cuda")
    big = _flat(W.config5())                     # 8^6 = 262144 cells > ZMC_STATIC_MAX_CELLS
    with pytest.raises(B.ZmcError) as ei:
        _static_path(big, out)
    assert ei.value.status == B.ERR_CAPACITY and "ZMC_STATIC_MAX_CELLS (4096)" in str(ei.value), str(ei.value)
    many_trials = _flat(W.config2()).with_(trials=33)      # 4096 cells * 33 trials > ZMC_STATIC_MAX_UNITS
    with pytest.raises(B.ZmcError) as ei:
        _static_path(many_trials, out)
    assert ei.value.status == B.ERR_CAPACITY and "ZMC_STATIC_MAX_UNITS (131072)" in str(ei.value), str(ei.value)
    with pytest.raises(B.ZmcError) as ei:        # dimensions without a pre-compiled kernel would need NVRTC, which allocates
        B.flat_static(13, (0.0,) * 13, (1.0,) * 13, 1, 100, 2, 1, B.SIN_SUM, None, B.F32, B.MATH_EXACT, out.data_ptr())
    assert ei.value.status == B.ERR_RANGE
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [-7.0, -7.0]    # nothing was launched
