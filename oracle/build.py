"""Build the ORACLE shared library (test infrastructure, not the product).

    python -m oracle.build

g++ -O2 -std=c++17 -ffp-contract=off -mfma: no implicit contraction, std::fmaf is
one instruction. The oracle is never tuned beyond this.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "zmc_oracle.cpp")
SRC_VEC = os.path.join(HERE, "zmc_oracle_vec.cpp")      # R15: vector-valued user integrands, on top of the public primitives
LIB = os.path.join(HERE, "libzmc_oracle.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-mfma", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    deps = [SRC, SRC_VEC, os.path.join(HERE, "zmc_oracle.h"), os.path.abspath(__file__)]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["g++", *FLAGS, "-o", LIB, SRC, SRC_VEC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
