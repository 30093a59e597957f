"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not the product).

g++ -O2 -ffp-contract=off: no fused multiply-adds, so the oracle's arithmetic is the one
written in gp_oracle.cpp.  -fcx-limited-range: plain textbook complex multiply/divide for
the complex-step derivatives (no libgcc inf/nan recovery paths).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gp_oracle.cpp")
LIB = os.path.join(HERE, "libgp_oracle.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "gp_oracle.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fcx-limited-range", "-fopenmp",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
