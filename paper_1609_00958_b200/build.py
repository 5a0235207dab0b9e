"""Builds libfp.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1609_00958_b200.build [--force]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfp.so")
SOURCES = [os.path.join(CSRC, "fp.cu")]
HEADERS = [os.path.join(CSRC, "fp_kernels.cuh"), os.path.join(CSRC, "fp_setup.cuh"),
           os.path.join(CSRC, "fp_aligned.cuh"), os.path.join(CSRC, "fp_tma.cuh"), os.path.join(CSRC, "fp_tex.cuh"), os.path.join(CSRC, "fp_probe.cuh"), os.path.join(CSRC, "fp_tile.cuh"), os.path.join(CSRC, "fp_bp.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "fp.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--fmad=true",            # fp32 sampling loop may contract; the fp64 set-up uses explicit _rn intrinsics
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc(), *NVCC_FLAGS, "-o", tmp, *SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
