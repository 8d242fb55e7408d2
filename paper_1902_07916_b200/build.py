"""Build libzmc.so (the product's C-ABI library, include/zmc.h) in-tree for sm_100a.

    python -m paper_1902_07916_b200.build [--force] [--verbose]

Steps
  1. csrc/zmc_device.cuh -> csrc/zmc_device_src.inc (the same text as a C++ raw string literal,
     handed to NVRTC at run time for user integrands and for 12 < D <= 16);
  2. nvcc -c, in parallel: zmc_lib.cu, zmc_static.cu and zmc_inst.cu once per pre-compiled
     (precision, math mode, integrand) combination;
  3. nvcc -shared -cudart static -> paper_1902_07916_b200/libzmc.so.
Flags: -gencode arch=compute_100a,code=sm_100a (B200 only), -lineinfo (ncu source pages),
--fmad=false (every fused multiply-add in the device code is written explicitly; R8).
nvcc cross-compiles without a GPU, so this runs in the CPU-only build container too.
"""
import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libzmc.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH + ["-O3", "-std=c++17", "-lineinfo", "--fmad=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2",
                     "-Xptxas", "-v"]

# (precision, mode, integrand id): must match zmc_inst.h / aot_lookup in zmc_lib.cu
COMBOS = [(0, 0, 0), (0, 0, 1), (0, 0, 2), (0, 0, 3),
          (1, 0, 0), (1, 0, 1), (1, 0, 2), (1, 0, 3),
          (1, 1, 2), (1, 1, 3)]


def _write_source_inc() -> str:
    src = open(os.path.join(CSRC, "zmc_device.cuh")).read()
    delim = "ZMCSRC"
    assert ")" + delim + '"' not in src
    # a raw string literal may not exceed the compiler's limit in one piece on some hosts: split on lines
    lines = src.splitlines(keepends=True)
    chunks, cur, size = [], [], 0
    for ln in lines:
        cur.append(ln)
        size += len(ln)
        if size > 8000:
            chunks.append("".join(cur))
            cur, size = [], 0
    if cur:
        chunks.append("".join(cur))
    text = "\n".join('R"%s(%s)%s"' % (delim, c, delim) for c in chunks) + "\n"
    out = os.path.join(CSRC, "zmc_device_src.inc")
    if not os.path.exists(out) or open(out).read() != text:
        with open(out, "w") as f:
            f.write(text)
    return out


def _sources():
    jobs = [("zmc_lib", os.path.join(CSRC, "zmc_lib.cu"), []),
            ("zmc_static", os.path.join(CSRC, "zmc_static.cu"), [])]      # zmc_flat_static: the entry point that allocates nothing
    for p, m, i in COMBOS:
        jobs.append(("zmc_inst_%d_%d_%d" % (p, m, i), os.path.join(CSRC, "zmc_inst.cu"),
                     ["-DZMC_INST_PREC=%d" % p, "-DZMC_INST_MODE=%d" % m, "-DZMC_INST_ID=%d" % i]))
    return jobs


def _stamp() -> str:
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".h")):
            h.update(name.encode())
            h.update(open(os.path.join(CSRC, name), "rb").read())
    h.update(open(os.path.join(os.path.dirname(HERE), "include", "zmc.h"), "rb").read())
    h.update(open(os.path.abspath(__file__), "rb").read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def is_current() -> bool:
    """True if libzmc.so was built from exactly these sources and flags."""
    stamp_file = os.path.join(OBJ, "stamp.txt")
    return os.path.exists(LIB) and os.path.exists(stamp_file) and open(stamp_file).read() == _stamp()


def _compile(job, verbose):
    name, src, defs = job
    obj = os.path.join(OBJ, name + ".o")
    cmd = [NVCC, *NVCC_FLAGS, *defs, "-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(os.path.join(OBJ, name + ".ptxas.txt"), "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (name, " ".join(cmd), r.stderr[-6000:]))
    if verbose:
        print("compiled", name)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile (if the sources changed) and return the path of libzmc.so."""
    os.makedirs(OBJ, exist_ok=True)
    _write_source_inc()
    stamp_file = os.path.join(OBJ, "stamp.txt")
    stamp = _stamp()
    if not force and os.path.exists(LIB) and os.path.exists(stamp_file) and open(stamp_file).read() == stamp:
        return LIB
    if not os.path.exists(NVCC):
        raise RuntimeError("nvcc not found at %s and libzmc.so is missing or stale" % NVCC)
    jobs = _sources()
    with cf.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(lambda j: _compile(j, verbose), jobs))
    cmd = [NVCC, *ARCH, "-shared", "-cudart", "static", "-o", LIB, *objs, "-ldl"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (" ".join(cmd), r.stderr[-6000:]))
    with open(stamp_file, "w") as f:
        f.write(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
