"""Build paper_2603_09528_b200/libtpt.so (the C-ABI library of include/tpt.h) with nvcc for sm_100a.

Usage: python -m paper_2603_09528_b200.build [--force] [--verbose]
nvcc cross-compiles without a GPU.  The library is built IN-TREE (it is git-ignored but travels to the
GPU box with the repo snapshot).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libtpt.so")
SOURCES = ["api.cu", "kernels.cu", "gemm_tma.cu", "thomas_onchip.cu", "projection.cu", "fft.cu", "plan_host.cpp"]
HEADERS = [os.path.join(CSRC, "kernels.cuh"), os.path.join(CSRC, "ptx.cuh"), os.path.join(CSRC, "tmap.hpp"), os.path.join(CSRC, "plan_host.hpp"), os.path.join(ROOT, "include", "tpt.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-fopenmp,-O3",
    "-shared",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")
    return exe


def is_fresh() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return all(os.path.getmtime(d) <= t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if is_fresh() and not force:
        return LIB
    cmd = [nvcc(), *NVCC_FLAGS]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES] + ["-lgomp"]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
