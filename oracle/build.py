"""Build oracle/liboracle.so (test infrastructure; see cdc_oracle.c header)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cdc_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")
FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-D_GNU_SOURCE", "-Wall", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    subprocess.check_call(["gcc", *FLAGS, "-o", LIB, SRC, "-lm"])
    return LIB


FAST_LIB = os.path.join(HERE, "liboracle_fast.so")
FAST_FLAGS = ["-O3", "-march=native", "-ffp-contract=fast", "-std=c11", "-D_GNU_SOURCE", "-shared", "-fPIC"]


def build_fast(force: bool = False) -> str:
    """The same source built for speed (timing only: bench.py reports it beside the parity build's number; no parity
    test ever loads it -- contraction changes the last bits)."""
    if not force and os.path.exists(FAST_LIB) and os.path.getmtime(FAST_LIB) >= os.path.getmtime(SRC):
        return FAST_LIB
    subprocess.check_call(["gcc", *FAST_FLAGS, "-o", FAST_LIB, SRC, "-lm"])
    return FAST_LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
