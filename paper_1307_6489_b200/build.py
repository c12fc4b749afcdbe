"""Build librta.so (the C-ABI library of include/rta.h) in-tree with nvcc for
sm_100a. ``python -m paper_1307_6489_b200.build`` or ``build()``."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librta.so")
SOURCES = [os.path.join(CSRC, "rta_kernels.cu"), os.path.join(CSRC, "rta_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "rta_internal.h"), os.path.join(ROOT, "include", "rta.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
]


def stale() -> bool:
    return (not os.path.exists(LIB)
            or any(os.path.getmtime(LIB) < os.path.getmtime(d) for d in DEPS))


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = ["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
