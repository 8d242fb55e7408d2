"""CPU-side checks of the boundary (no compute calls): libzmc.so builds for sm_100a, loads, exports every
symbol include/zmc.h declares, validates arguments, and refuses to work without a CUDA device
(there is no CPU fallback; the oracle is never reachable from the product)."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

from paper_1902_07916_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "zmc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(zmc_[a-z_]+)\s*\(", text)))


def test_header_symbols_all_exported():
    L = B.lib()
    names = _declared()
    assert set(names) == set(B.EXPORTS), (names, B.EXPORTS)
    for n in names:
        assert getattr(L, n) is not None


def test_library_is_sm100a_only_and_has_no_oracle_symbols():
    out = subprocess.run(["cuobjdump", "-lelf", B.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs
    syms = subprocess.run(["nm", "-D", "--defined-only", B.LIB_PATH], capture_output=True, text=True).stdout
    assert "orc_" not in syms
    # the product never imports the oracle
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1902_07916_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "zmc_oracle" not in src, f


def test_create_validates_arguments():
    L = B.lib()
    lo = np.zeros(3)
    up = np.ones(3)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))

    def create(dim=3, lower=lo, upper=up, g=4, N=100, T=5, depth=2, m=1.5, seed=1):
        h = C.c_void_p(0xDEAD)     # a failed zmc_create must overwrite this with NULL: there is nothing to destroy
        rc = L.zmc_create(C.byref(h), dim, dp(lower) if lower is not None else None, dp(upper) if upper is not None else None,
                          g, N, T, depth, m, seed)
        assert rc != B.OK          # every case below is invalid (and without a device even a valid one fails)
        assert not h, "a failed zmc_create left a context behind"
        return rc, L.zmc_last_error(None).decode()

    assert create(dim=0)[0] == B.ERR_ARG
    assert create(lower=None)[0] == B.ERR_ARG
    assert create(g=0)[0] == B.ERR_ARG
    assert create(N=0)[0] == B.ERR_ARG
    assert create(T=0)[0] == B.ERR_ARG
    assert create(depth=0)[0] == B.ERR_ARG
    assert create(m=float("nan"))[0] == B.ERR_ARG
    assert create(upper=np.array([1.0, 0.0, 1.0]))[0] == B.ERR_ARG
    assert create(upper=np.array([1.0, np.inf, 1.0]))[0] == B.ERR_ARG
    rc, msg = create(T=256)
    assert rc == B.ERR_RANGE and "255" in msg
    assert create(depth=16)[0] == B.ERR_RANGE
    assert create(dim=17, lower=np.zeros(17), upper=np.ones(17))[0] == B.ERR_RANGE
    assert create(N=2 ** 33)[0] == B.ERR_RANGE                          # N*D >= 2^34 - 2^14 (R3)
    rc, msg = create(dim=1, lower=np.zeros(1), upper=np.ones(1), N=2 ** 34 - 2 ** 14)
    assert rc == B.ERR_RANGE and "2^34 - 2^14" in msg
    assert create(dim=12, lower=np.zeros(12), upper=np.ones(12), g=4, depth=4)[0] == B.ERR_RANGE   # 96-bit path
    assert create(g=70000, depth=2)[0] == B.ERR_RANGE                   # g^depth > 2^32
    assert L.zmc_create(None, 3, dp(lo), dp(up), 4, 100, 5, 2, 1.5, 1) == B.ERR_ARG
    assert L.zmc_last_error(None).decode() == "out is null"
    assert L.zmc_status_string(B.ERR_CAPACITY).decode() == "level capacity exceeded"


def test_no_device_means_error_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(B.ZmcError) as e:
        B.Integrator(3, [0.0] * 3, [1.0] * 3, 4, 100, 5, 2, 1.5, 1)
    assert e.value.status == B.ERR_CUDA and "no CUDA device" in str(e.value)


def test_headline_kernels_keep_their_register_budget():
    """The sampling kernel's speed hangs on ptxas' schedule (profiles/r1_variants.md: a three-line change once cost 30 registers
    and 4 %). The build keeps ptxas -v per translation unit: the headline instances must stay within the register count that
    gives them 4 CTAs per SM, without spills."""
    from paper_1902_07916_b200 import build as zbuild
    B.lib()
    budget = {   # (integrand id, D) of FP32 exact-mode UKEY kernels -> registers for 4 CTAs of 128 threads per SM
        ("zmc_inst_1_0_2", "ZmcIntegrandILi2ELi6ELi1ELi0EELb1ELb0"): 128,     # sin 6-D: configs 2 and 5
        ("zmc_inst_1_0_3", "ZmcIntegrandILi3ELi9ELi1ELi0EELb1ELb0"): 128,     # Gaussian 9-D: config 3
        ("zmc_inst_1_0_3", "ZmcIntegrandILi3ELi12ELi1ELi0EELb1ELb0"): 128,    # Gaussian 12-D: paper Table 4
        ("zmc_inst_1_0_3", "ZmcIntegrandILi3ELi4ELi1ELi0EELb0ELb0"): 102,     # Gaussian 4-D, per-item key: config 4 (5 CTAs)
    }
    for (unit, key), limit in budget.items():
        path = os.path.join(zbuild.OBJ, unit + ".ptxas.txt")
        if not os.path.exists(path):
            pytest.skip("no ptxas log (library not built here)")
        lines = open(path).read().splitlines()
        idx = [i for i, l in enumerate(lines) if "Compiling entry function" in l and "zmc_sample_kernel" in l and key in l]
        assert len(idx) == 1, (unit, key, len(idx))
        block = " ".join(lines[idx[0]: idx[0] + 4])
        regs = int(re.search(r"Used (\d+) registers", block).group(1))
        assert regs <= limit, (key, regs, limit)
        assert "0 bytes spill stores" in block, block


def test_binding_constants_match_the_header():
    """Every enumerator of include/zmc.h that the ctypes binding mirrors has the same value there, and the ctypes
    structures have the size the C compiler gives them."""
    text = open(os.path.join(ROOT, "include", "zmc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    enums = {k: int(v) for k, v in re.findall(r"\b(ZMC_[A-Z0-9_]+)\s*=\s*(-?\d+)", text)}
    mirror = {
        "ZMC_OK": B.OK, "ZMC_ERR_ARG": B.ERR_ARG, "ZMC_ERR_RANGE": B.ERR_RANGE, "ZMC_ERR_NO_INTEGRAND": B.ERR_NO_INTEGRAND,
        "ZMC_ERR_COMPILE": B.ERR_COMPILE, "ZMC_ERR_CUDA": B.ERR_CUDA, "ZMC_ERR_CAPACITY": B.ERR_CAPACITY,
        "ZMC_ERR_NOT_RUN": B.ERR_NOT_RUN, "ZMC_ERR_STATE": B.ERR_STATE,
        "ZMC_CONST": B.CONST, "ZMC_LINEAR": B.LINEAR, "ZMC_SIN_SUM": B.SIN_SUM, "ZMC_EXP_QUAD": B.EXP_QUAD, "ZMC_USER": B.USER,
        "ZMC_OPT_PRECISION": B.OPT_PRECISION, "ZMC_OPT_MATH": B.OPT_MATH, "ZMC_OPT_MAX_GROUPS_PER_LEVEL": B.OPT_MAX_GROUPS_PER_LEVEL,
        "ZMC_OPT_KEEP_LEVEL_STATS": B.OPT_KEEP_LEVEL_STATS, "ZMC_OPT_MAX_CELLS_PER_LEVEL": B.OPT_MAX_CELLS_PER_LEVEL,
        "ZMC_OPT_GRID_BLOCKS": B.OPT_GRID_BLOCKS, "ZMC_OPT_TARGET_ITEMS": B.OPT_TARGET_ITEMS, "ZMC_OPT_USE_GRAPH": B.OPT_USE_GRAPH,
        "ZMC_OPT_SPREAD": B.OPT_SPREAD, "ZMC_OPT_BUDGET_ORDER": B.OPT_BUDGET_ORDER, "ZMC_OPT_SINGLE_LAUNCH": B.OPT_SINGLE_LAUNCH,
        "ZMC_F64": B.F64, "ZMC_F32": B.F32, "ZMC_MATH_EXACT": B.MATH_EXACT, "ZMC_MATH_FAST": B.MATH_FAST,
        "ZMC_SPREAD_TRIALS": B.SPREAD_TRIALS, "ZMC_SPREAD_SAMPLES": B.SPREAD_SAMPLES,
        "ZMC_BUDGET_PATH_ORDER": B.BUDGET_PATH_ORDER, "ZMC_BUDGET_LARGEST_SPREAD": B.BUDGET_LARGEST_SPREAD,
    }
    for name, value in mirror.items():
        assert enums[name] == value, name
    # the fixed limits of zmc_flat_static are #defines
    defs = dict(re.findall(r"#define\s+(ZMC_STATIC_[A-Z_]+)\s+(.+)", text))
    assert eval(defs["ZMC_STATIC_SCRATCH_BYTES"].replace("u", "")) == B.STATIC_SCRATCH_BYTES
    assert int(defs["ZMC_STATIC_MAX_CELLS"]) == B.STATIC_MAX_CELLS and int(defs["ZMC_STATIC_MAX_UNITS"]) == B.STATIC_MAX_UNITS
    assert int(defs["ZMC_STATIC_MAX_PARAMS"]) == B.STATIC_MAX_PARAMS
    assert int(re.search(r"#define ZMC_MAX_DEPTH (\d+)", text).group(1)) == B.MAX_DEPTH
    # struct sizes as the C compiler sees them
    src = '#include <stdio.h>\n#include "zmc.h"\nint main(void) { printf("%zu %zu\\n", sizeof(zmc_level_stats), sizeof(zmc_stats_t)); return 0; }\n'
    import tempfile
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "s.c"), "w").write(src)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(d, "s"), os.path.join(d, "s.c")], check=True)
        a, b = subprocess.run([os.path.join(d, "s")], capture_output=True, text=True, check=True).stdout.split()
    assert int(a) == C.sizeof(B.LevelStats) and int(b) == C.sizeof(B.Stats)


def test_failed_create_from_c_leaves_nothing_to_destroy():
    """The contract of include/zmc.h as a C caller sees it: a failed zmc_create sets *out to NULL, the reason is
    zmc_last_error(NULL), zmc_destroy(NULL) is a no-op, and every other call refuses a NULL context."""
    src = r"""
#include <stdio.h>
#include <string.h>
#include "zmc.h"
int main(void) {
    double lo[3] = {0, 0, 0}, up[3] = {1, 1, 1}, bad_up[3] = {1, 0, 1};
    zmc_ctx* c = (zmc_ctx*)0x1;
    int rc = zmc_create(&c, 3, lo, bad_up, 4, 100, 5, 2, 1.5, 1);
    if (rc != ZMC_ERR_ARG || c != NULL) { printf("bounds: rc %d ctx %p\n", rc, (void*)c); return 1; }
    if (strstr(zmc_last_error(NULL), "upper > lower") == NULL) { printf("message: %s\n", zmc_last_error(NULL)); return 2; }
    c = (zmc_ctx*)0x1;
    rc = zmc_create(&c, 3, lo, up, 4, 100, 300, 2, 1.5, 1);
    if (rc != ZMC_ERR_RANGE || c != NULL) { printf("trials: rc %d ctx %p\n", rc, (void*)c); return 3; }
    zmc_destroy(c);   /* NULL: no-op */
    if (zmc_run(NULL, NULL) != ZMC_ERR_ARG || zmc_set_option(NULL, ZMC_OPT_PRECISION, ZMC_F32) != ZMC_ERR_ARG) return 4;
    double v, s;
    if (zmc_result(NULL, &v, &s) != ZMC_ERR_ARG) return 5;
    printf("ok\n");
    return 0;
}
"""
    import tempfile
    B.lib()
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "t.c"), "w").write(src)
        exe = os.path.join(d, "t")
        subprocess.run(["gcc", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", exe, os.path.join(d, "t.c"),
                        B.LIB_PATH, "-Wl,-rpath," + os.path.dirname(B.LIB_PATH)], check=True)
        r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0 and r.stdout.strip() == "ok", (r.returncode, r.stdout, r.stderr)


def test_microbench_is_not_part_of_the_product_library():
    syms = subprocess.run(["nm", "-D", "--defined-only", B.LIB_PATH], capture_output=True, text=True).stdout
    assert "zmc_microbench" not in syms
    assert "zmc_microbench" not in open(os.path.join(ROOT, "include", "zmc.h")).read()
