"""Build libgeo.so (the C-ABI library of include/geo.h) for sm_100a, in-tree.

    python -m paper_1803_08320_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
working-tree snapshot.  Flags: -O3 -lineinfo (ncu source page), default -fmad (FMA contraction is
part of the design), no fast-math.
"""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libgeo.so")
SOURCES = [os.path.join(CSRC, "geo_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "geo_kernel.cuh"), os.path.join(CSRC, "geo_rhs.cuh"),
                  os.path.join(CSRC, "geo_rk45.cuh"), os.path.join(CSRC, "geo_tab.cuh"), os.path.join(CSRC, "geo_tabg.cuh"),
                  os.path.join(CSRC, "geo_ks.cuh"), os.path.join(CSRC, "geo_ks_rk45.cuh"),
                  os.path.join(ROOT, "include", "geo.h"), os.path.join(ROOT, "include", "geo_dev.h")]


def nvcc_path() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = f"{LIB}.tmp{os.getpid()}"      # several ranks may build at once: private file, atomic rename
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
           "-Xcompiler", "-fPIC,-Wall", "-shared", "-I", os.path.join(ROOT, "include"),
           "-o", tmp] + SOURCES
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
