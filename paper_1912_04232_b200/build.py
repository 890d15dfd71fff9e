"""Build libmd_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = [os.path.join(HERE, "csrc", "md.cu")]
DEPS = SRC + [os.path.join(HERE, "csrc", "md_kernels.cuh"),
              os.path.join(HERE, "csrc", "md_force32.cuh"),
              os.path.join(HERE, "csrc", "md_nbr2.cuh"),
              os.path.join(HERE, "csrc", "md_fire.cuh"),
              os.path.join(HERE, "csrc", "md_brownian.cuh"),
              os.path.join(HERE, "csrc", "md_nh.cuh"), os.path.join(HERE, "csrc", "md_flock.cuh"), os.path.join(ROOT, "include", "md.h")]
LIB = os.environ.get("MD_B200_LIB") or os.path.join(HERE, "libmd_b200.so")   # override: a variant build

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"),
    "-I", os.path.join(HERE, "csrc"),
]


def nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        extra = os.environ.get("MD_B200_NVCC_EXTRA", "").split()      # e.g. -DMD_F32_U=8 (tuning builds)
        cmd = [nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SRC
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
