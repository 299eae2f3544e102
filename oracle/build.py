"""Build the oracle shared library (test infrastructure). g++ -O2 -ffp-contract=off, single thread."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libswe_ref.so")
SRC = [os.path.join(HERE, "swe_ref.cpp")]
DEPS = SRC + [os.path.join(HERE, "swe_ref.h")]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB] + SRC
    subprocess.run(cmd, check=True)
    return LIB


LIB_F32 = os.path.join(HERE, "libswe_ref_f32.so")


def build_f32(force: bool = False) -> str:
    """The same source with -DSWE_REF_REAL=float: the single-precision oracle."""
    if not force and os.path.exists(LIB_F32) and all(os.path.getmtime(LIB_F32) >= os.path.getmtime(d) for d in DEPS):
        return LIB_F32
    cmd = ["g++", "-std=c++17", "-O2", "-DSWE_REF_REAL=float", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-Wdouble-promotion", "-o", LIB_F32] + SRC
    subprocess.run(cmd, check=True)
    return LIB_F32


LIB_OMP = os.path.join(HERE, "libswe_ref_omp.so")


def build_omp(force: bool = False) -> str:
    """The same source with -fopenmp -DSWE_REF_OMP: bench.py's optional cpu_baseline_omp line (the
    paper's `omp` backend).  No test uses it."""
    if not force and os.path.exists(LIB_OMP) and all(os.path.getmtime(LIB_OMP) >= os.path.getmtime(d) for d in DEPS):
        return LIB_OMP
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-DSWE_REF_OMP", "-ffp-contract=off", "-fno-fast-math", "-fPIC",
           "-shared", "-Wall", "-Wextra", "-o", LIB_OMP] + SRC
    subprocess.run(cmd, check=True)
    return LIB_OMP


if __name__ == "__main__":
    print(build(force=True))
