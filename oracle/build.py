"""Builds the CPU oracle (oracle/cgks_ref.c) into oracle/libcgks_ref.so.  TEST INFRASTRUCTURE ONLY.

-ffp-contract=off keeps gcc from fusing multiply-adds, so the oracle's rounding is the plain
IEEE sequence of the formulas as written (tolerance derivation).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cgks_ref.c")
LIB = os.path.join(HERE, "libcgks_ref.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "cgks_ref.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wno-unused-variable", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
