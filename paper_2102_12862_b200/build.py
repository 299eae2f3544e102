"""Build libswe_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2102_12862_b200.build [--force]

-fmad=false / -ffp-contract=off: the arithmetic contract of DESIGN.md R-14 (no FMA contraction on either side).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libswe_b200.so")
OBJ = os.path.join(HERE, "build")
# swe_abi.cu: the C-ABI and every kernel but the fused patch step; swe_static.cu: the entry point that allocates nothing; swe_patch_t*.cu: the instances of the fused patch kernel,
# one translation unit per block size -- compiled in parallel (the kernel is ~5000 SASS instructions, ~50 instances)
SRC = [os.path.join(CSRC, "swe_abi.cu"), os.path.join(CSRC, "swe_static.cu")] + [os.path.join(CSRC, f"swe_patch_t{t}.cu") for t in (32, 64, 128, 192, 256, 384, 512, 1024)]
DEPS = SRC + [os.path.join(CSRC, f) for f in ("swe_kernels.cuh", "swe_patch2_kernel.cuh", "swe_patch_inst.cuh", "swe_cbrt.cuh",
                                              "swe_types.h", "mesh_prep.hpp", "patch_blob.hpp")] + [
    os.path.join(os.path.dirname(HERE), "include", "swe.h")]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-fmad=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math,-Wall",
]


def nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJ, exist_ok=True)
    objs = [os.path.join(OBJ, os.path.basename(s)[:-3] + ".o") for s in SRC]

    def compile_one(pair):
        src, obj = pair
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
        subprocess.run(cmd, check=True)

    with ThreadPoolExecutor(max_workers=min(len(SRC), os.cpu_count() or 4)) as pool:
        list(pool.map(compile_one, zip(SRC, objs)))
    subprocess.run([nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
