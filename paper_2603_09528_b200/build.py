"""Build paper_2603_09528_b200/libtpt.so (the C-ABI library of include/tpt.h) with nvcc for sm_100a.

Usage: python -m paper_2603_09528_b200.build [--force] [--verbose]
nvcc cross-compiles without a GPU.  The library is built IN-TREE (it is git-ignored but travels to the
GPU box with the repo snapshot).  Each source is compiled to its own object (in parallel, only when stale) under
paper_2603_09528_b200/build/, then linked.
"""
from __future__ import annotations

import concurrent.futures
import os
import shutil
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
OBJ = os.path.join(PKG, "build")
LIB = os.path.join(PKG, "libtpt.so")
SOURCES = ["api.cu", "kernels.cu", "gemm_tma.cu", "thomas_onchip.cu", "projection.cu", "fft.cu", "plan_host.cpp",
           "sharded.cu", "fused_small.cu"]
HEADERS = [os.path.join(CSRC, h) for h in ("kernels.cuh", "ptx.cuh", "tmap.hpp", "plan_host.hpp", "devonce.hpp", "plan.hpp")] + \
          [os.path.join(ROOT, "include", "tpt.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-fopenmp,-O3",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")
    return exe


def _sources():
    return [s for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]


def _deps_mtime() -> float:
    deps = [h for h in HEADERS if os.path.exists(h)] + [os.path.abspath(__file__)]
    return max(os.path.getmtime(d) for d in deps)


def is_fresh() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(os.path.join(CSRC, s)) <= t for s in _sources()) and _deps_mtime() <= t


def _compile(src: str, verbose: bool) -> str:
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    cmd = [nvcc(), *NVCC_FLAGS]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return res.stdout + res.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if is_fresh() and not force:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    hdr_t = _deps_mtime()
    stale = []
    for s in _sources():
        obj = os.path.join(OBJ, os.path.splitext(s)[0] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(hdr_t, os.path.getmtime(os.path.join(CSRC, s))):
            stale.append(s)
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, max(1, len(stale)))) as pool:
        logs = list(pool.map(lambda s: _compile(s, verbose), stale))
    if verbose:
        print("".join(logs))
    objs = [os.path.join(OBJ, os.path.splitext(s)[0] + ".o") for s in _sources()]
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-o", LIB, *objs, "-lgomp"]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
