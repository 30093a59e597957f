"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not the product).

g++ -O2 -ffp-contract=off: no fused multiply-adds, so the oracle's arithmetic is the one
written in gp_oracle.cpp.  -fcx-limited-range: plain textbook complex multiply/divide for
the complex-step derivatives (no libgcc inf/nan recovery paths).

build_rounding_probe() compiles the SAME source a second time with `-ffp-contract=fast -mfma`
into libgp_oracle_fma.so.  That library is not "the oracle": it exists only so that the parity
tests can measure, ray by ray, how far the oracle's own FP64 result moves when nothing but the
rounding of its arithmetic changes (R30).  Expected values always come
from the contraction-free build.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gp_oracle.cpp")
SRC_SHADE = os.path.join(HERE, "gp_shade_oracle.cpp")
LIB = os.path.join(HERE, "libgp_oracle.so")
LIB_FMA = os.path.join(HERE, "libgp_oracle_fma.so")
LIB_X87 = os.path.join(HERE, "libgp_oracle_x87.so")


def build(force: bool = False) -> str:
    deps = [SRC, SRC_SHADE, os.path.join(HERE, "gp_oracle.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fcx-limited-range", "-fopenmp",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC, SRC_SHADE]
    subprocess.check_call(cmd)
    return LIB


def build_rounding_probe(force: bool = False) -> str:
    deps = [SRC, SRC_SHADE, os.path.join(HERE, "gp_oracle.h")]
    if (not force and os.path.exists(LIB_FMA)
            and all(os.path.getmtime(LIB_FMA) >= os.path.getmtime(d) for d in deps)):
        return LIB_FMA
    with open("/proc/cpuinfo") as f:
        if " fma" not in f.read():
            raise RuntimeError("the rounding probe needs a host CPU with FMA instructions")
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=fast", "-mfma", "-fcx-limited-range",
           "-fopenmp", "-fPIC", "-shared", "-o", LIB_FMA, SRC, SRC_SHADE]
    subprocess.check_call(cmd)
    return LIB_FMA


def build_rounding_probe_x87(force: bool = False) -> str:
    """A third rounding sample of the same source: x87 arithmetic (64-bit mantissa in registers,
    rounded to double when stored).  Used by tests/test_parity_threshold.py only, to measure how far
    one more rounding sample can exceed the FMA probe's spread (the derivation of
    tests/parity_rules.py SENSITIVE_AT); never for expected values."""
    deps = [SRC, SRC_SHADE, os.path.join(HERE, "gp_oracle.h")]
    if (not force and os.path.exists(LIB_X87)
            and all(os.path.getmtime(LIB_X87) >= os.path.getmtime(d) for d in deps)):
        return LIB_X87
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-mfpmath=387", "-fcx-limited-range",
           "-fopenmp", "-fPIC", "-shared", "-o", LIB_X87, SRC, SRC_SHADE]
    subprocess.check_call(cmd)
    return LIB_X87


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
    print(build_rounding_probe(force="--force" in sys.argv))
