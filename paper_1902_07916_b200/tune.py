"""Variant sweep of the sampling kernel: what ZmcTune in csrc/zmc_device.cuh encodes (profiles/r1_variants.md).

    python -m paper_1902_07916_b200.tune --build          # nvcc, here or on the GPU box (csrc/build/tune/, ~100 small programs)
    python -m paper_1902_07916_b200.tune --run            # needs a B200: runs what was built, prints a markdown table

Each program is csrc/zmc_tune_main.cu + the committed zmc_device.cuh with one combination of
-DZMC_TUNE_PACKED={0,1} -DZMC_TUNE_UNROLL={2,4} -DZMC_TUNE_MINB={3,4} -DZMC_TUNE_P0ADD={0,2}; "committed" has no override.
All variants of a case must print the same checksum of the per-(cell, trial) sums.
"""
import concurrent.futures as cf
import itertools
import os
import re
import subprocess
import sys

from . import build as zbuild

CSRC = zbuild.CSRC
OUT = os.path.join(CSRC, "build", "tune")
CASES = {   # name -> -D flags selecting dimension / integrand / mode / key handling
    "sin6": "-DVD=6 -DVID=2",
    "gauss9": "-DVD=9 -DVID=3",
    "gauss12": "-DVD=12 -DVID=3",
    "gauss4_per_item_key": "-DVD=4 -DVID=3 -DVUKEY=false",
    "sin6_fast": "-DVD=6 -DVID=2 -DVMODE=1",
    "gauss9_fast": "-DVD=9 -DVID=3 -DVMODE=1",
}
GRID = list(itertools.product((0, 1), (2, 4), (3, 4), (0, 2)))


def variants(case):
    yield case + "__committed", ""
    for p, u, m, a in GRID:
        yield ("%s__p%du%dm%da%d" % (case, p, u, m, a),
               "-DZMC_TUNE_PACKED=%d -DZMC_TUNE_UNROLL=%d -DZMC_TUNE_MINB=%d -DZMC_TUNE_P0ADD=%d" % (p, u, m, a))


def _compile(job):
    name, flags = job
    exe = os.path.join(OUT, name)
    cmd = [zbuild.NVCC, *zbuild.ARCH, "-O3", "-std=c++17", "-lineinfo", "--fmad=false", "-I", CSRC,
           '-DVNAME="%s"' % name, *flags.split(), "-o", exe, os.path.join(CSRC, "zmc_tune_main.cu")]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s" % (name, r.stderr[-3000:]))
    return exe


def build(cases):
    os.makedirs(OUT, exist_ok=True)
    jobs = [(n, CASES[c] + " " + f) for c in cases for n, f in variants(c)]
    with cf.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        list(ex.map(_compile, jobs))
    print("built %d programs in %s" % (len(jobs), OUT))


def run(cases):
    pat = re.compile(r"regs=(\d+) occ=(\d+) .*?([\d.]+) ms\s+([\d.]+) Gevals/s\s+frac=([\d.]+)\s+chk=([0-9a-f]+)")
    for c in cases:
        rows, chks = [], set()
        for n, _ in variants(c):
            exe = os.path.join(OUT, n)
            if not os.path.exists(exe):
                continue
            out = subprocess.run([exe], capture_output=True, text=True).stdout
            m = pat.search(out)
            if not m:
                rows.append((n, None))
                continue
            regs, occ, ms, ge, frac, chk = m.groups()
            chks.add(chk)
            rows.append((n.split("__")[1], (int(regs), int(occ), float(ms), float(ge), float(frac))))
        print("\n### %s (checksums identical: %s)\n" % (c, "yes" if len(chks) == 1 else "NO " + str(chks)))
        print("| variant (p = packed, u = groups per trip, m = MINB, a = P0_ADD/CARRY) | registers | CTAs/SM | ms | Gevals/s | frac of the roof |")
        print("|---|---|---|---|---|---|")
        for n, v in sorted(rows, key=lambda r: -(r[1][4] if r[1] else 0)):
            print("| %s | %s |" % (n, " | ".join(str(x) for x in v) if v else "failed"))


if __name__ == "__main__":
    cases = [a for a in sys.argv[1:] if not a.startswith("--")] or list(CASES)
    if "--build" in sys.argv or "--run" not in sys.argv:
        build(cases)
    if "--run" in sys.argv:
        run(cases)
