"""Build the CPU oracle (test infrastructure) with gcc: oracle/liboracle_fredec.so.

One shared object holds the FP64 oracle (`oracle_*`) and the 80-bit long double build of
the same source (`oracle_*_ld`).  -fopenmp parallelises only the loop over grid
frequencies; `oracle_set_threads(1)` gives the single-threaded oracle.  No -ffast-math,
no FMA contraction: the arithmetic is exactly what oracle_fredec.c spells out.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle_fredec.c")
LIB = os.path.join(HERE, "liboracle_fredec.so")
CFLAGS = ["-O2", "-fPIC", "-fopenmp", "-ffp-contract=off", "-Wall", "-Wextra", "-std=c11"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(
            os.path.getmtime(SRC), os.path.getmtime(__file__)):
        return LIB
    obj_d = os.path.join(HERE, "oracle_fredec_f64.o")
    obj_ld = os.path.join(HERE, "oracle_fredec_f80.o")
    subprocess.check_call(["gcc", *CFLAGS, "-c", SRC, "-o", obj_d])
    subprocess.check_call(["gcc", *CFLAGS, "-DORACLE_REAL=long double", "-DORACLE_SUFFIX=_ld",
                           "-c", SRC, "-o", obj_ld])
    subprocess.check_call(["gcc", "-shared", "-fopenmp", obj_d, obj_ld, "-lm", "-o", LIB])
    return LIB


if __name__ == "__main__":
    print(build(force=True))
