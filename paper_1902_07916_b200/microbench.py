"""Issue-rate microbenchmarks of the pipes the sampling kernel uses (csrc/zmc_microbench.cu, built as its own
library libzmc_microbench.so by build.build_microbench(); a measurement tool, not part of the product ABI).

    python -m paper_1902_07916_b200.microbench            # prints a markdown table (needs a B200)
    python -m paper_1902_07916_b200.microbench --probe DIM INTEGRAND UKEY [-DNAME=VALUE ...] [-- n_inst g N T reps]
        # one level-1 launch of the sampling kernel instance (csrc/zmc_kernel_probe.cu, compiled on the spot with the given
        # macros): evaluations/s, fraction of the ALU roof, checksum. E.g. the per-item-key cost at D = 4:
        #   --probe 4 3 0 -- 256 6 4096 5 4      against      --probe 4 3 1 -- 256 6 4096 5 4

They give the denominator of the ALU roofline: warp-instructions per SM per clock
for IMAD.WIDE.U32, LOP3, FFMA, ... and whole Philox4x32-10 calls.
"""
import ctypes as C

from . import build as _build

_lib = None


class MicrobenchError(RuntimeError):
    def __init__(self, status):
        super().__init__("zmc_microbench status %d" % status)
        self.status = status


def microbench(which: int, stream: int = 0):
    """which: 0 IMAD.WIDE.U32, 1 LOP3, 2 IMAD.WIDE+LOP3, 3 FFMA, 4 FADD, 5 DADD, 6 F2F pair, 7 MUFU.SIN, 8 MUFU.EX2, 9 DFMA,
    10 Philox4x32-10 calls, 11 I2F/F2I pair, 12 LEA.HI, 13 IMAD lo, 14 IMAD.HI, 15 64-bit add, 16 IMAD.WIDE by a register;
    100 + 10*X + j: Philox calls each followed by K = (0, 10, 20, 40)[j] extra instructions of kind X (see MIX).
    Returns (warp-instructions per SM per clock, SM MHz seen)."""
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build_microbench())
        _lib.zmc_microbench.argtypes = [C.c_int, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    r, mhz = C.c_double(), C.c_double()
    rc = _lib.zmc_microbench(which, C.c_void_p(stream), C.byref(r), C.byref(mhz))
    if rc != 0:
        raise MicrobenchError(rc)
    return r.value, mhz.value

NAMES = {0: "IMAD.WIDE.U32", 1: "LOP3", 2: "IMAD.WIDE.U32 + LOP3 (Philox round mix)", 3: "FFMA", 4: "FADD", 5: "DADD",
         6: "F2F.F64.F32 + F2F.F32.F64 (dependent pair, per instruction)", 7: "MUFU.SIN", 8: "MUFU.EX2", 9: "DFMA", 10: "Philox4x32-10 calls (x32 lanes)",
         11: "I2F.F64.U32 + F2I.U32.F64 (dependent pair, per instruction)", 12: "LEA.HI-like (shr + or)", 13: "IMAD.U32 lo", 14: "IMAD.HI.U32",
         15: "IADD3 + IADD3.X (64-bit add)", 16: "IMAD.WIDE.U32 with register multiplier"}


def main():
    print("| which | instruction | warp-instr / SM / clk | clocks per warp-instr per sub-partition | SM MHz |")
    print("|---|---|---|---|---|")
    for w in sorted(NAMES):
        try:
            r, mhz = microbench(w)
        except MicrobenchError as e:
            print("| %d | %s | error %d | | |" % (w, NAMES[w], e.status))
            continue
        print("| %d | %s | %.3f | %.2f | %.0f |" % (w, NAMES[w], r, 4.0 / r if r > 0 else float("nan"), mhz))


MIX = {1: "LOP3", 2: "FFMA", 3: "FADD", 4: "DADD", 5: "FFMA2", 6: "IMAD (lo)", 7: "SHF"}
MIX_K = (0, 10, 20, 40)


def mix_table():
    """Clocks per Philox call per sub-partition with K extra instructions of one kind after each call, and the slope
    = what one more instruction of that kind costs next to the generator (the dispatch-slot model of DESIGN.md 6)."""
    print()
    print("| extra instruction | " + " | ".join("K=%d" % k for k in MIX_K) + " | clocks per extra instruction (K=40 vs K=0) |")
    print("|---|" + "---|" * (len(MIX_K) + 1))
    for x in sorted(MIX):
        clk = []
        for j, k in enumerate(MIX_K):
            r, _ = microbench(100 + 10 * x + j)
            clk.append(4.0 / r)
        print("| %s | " % MIX[x] + " | ".join("%.1f" % c for c in clk) + " | %.2f |" % ((clk[-1] - clk[0]) / MIX_K[-1]))


def probe(argv):
    """Compile csrc/zmc_kernel_probe.cu for one kernel instance (nvcc, sm_100a, the product's flags) and run it."""
    import os
    import subprocess
    import tempfile
    run_args = []
    if "--" in argv:
        i = argv.index("--")
        argv, run_args = argv[:i], argv[i + 1:]
    dim, integrand, ukey = argv[0], argv[1], argv[2]
    defs = ["-DTD=%s" % dim, "-DTID=%s" % integrand, "-DTUKEY=%s" % ukey] + list(argv[3:])
    exe = os.path.join(tempfile.gettempdir(), "zmc_kernel_probe_%d" % os.getpid())
    cmd = [_build.NVCC, *_build.ARCH, "-O3", "-std=c++17", "--fmad=false", "-lineinfo", "-diag-suppress", "550", "-Xptxas", "-v",
           *defs, "-I", _build.CSRC, os.path.join(_build.CSRC, "zmc_kernel_probe.cu"), "-o", exe]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), r.stderr[-4000:]))
    regs = [ln.strip() for ln in r.stderr.splitlines() if "registers" in ln]
    print(" ".join(defs), "|", regs[0] if regs else "", flush=True)
    try:
        subprocess.run([exe, *run_args], check=True)
    finally:
        os.unlink(exe)


if __name__ == "__main__":
    import sys
    if len(sys.argv) > 1 and sys.argv[1] == "--probe":
        probe(sys.argv[2:])
    else:
        main()
        mix_table()
