"""Build oracle/libtpt_oracle.so from tpt_oracle.c with gcc.  TEST INFRASTRUCTURE (see tpt_oracle.h).

Usage: python oracle/build.py [--force]
The flags are fixed (no -march=native: the .so travels to another machine); if the host CPU lacks
AVX2/FMA the generic fallback is used.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tpt_oracle.c")
HDR = os.path.join(HERE, "tpt_oracle.h")
LIB = os.path.join(HERE, "libtpt_oracle.so")
FLAGFILE = os.path.join(HERE, ".libtpt_oracle.flags")


def _cpu_has_avx2_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    flags = set(line.split(":", 1)[1].split())
                    return "avx2" in flags and "fma" in flags
    except OSError:
        pass
    return False


def flags() -> list:
    base = ["-O3", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-math-errno", "-Wall", "-Wextra"]
    if _cpu_has_avx2_fma():
        base += ["-mavx2", "-mfma"]
    return base


def build(force: bool = False) -> str:
    fl = flags()
    stamp = " ".join(fl)
    fresh = (
        os.path.exists(LIB)
        and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        and os.path.exists(FLAGFILE)
        and open(FLAGFILE).read() == stamp
    )
    if fresh and not force:
        return LIB
    cmd = ["gcc", *fl, "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    with open(FLAGFILE, "w") as fh:
        fh.write(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
