"""Build librta.so (the C-ABI library of include/rta.h) in-tree with nvcc for
sm_100a, and beside it librta_testing.so: the same objects with rta_api.cu
compiled -DRTA_TESTING, which adds the test hooks (rta_debug_*, *_generic) that
the shipped library does not export. ``python -m paper_1307_6489_b200.build``
or ``build()``."""
from __future__ import annotations

import os
import shlex
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librta.so")
TEST_LIB = os.path.join(HERE, "librta_testing.so")
SOURCES = [os.path.join(CSRC, n) for n in ("rta_kernels.cu", "rta_image.cu", "rta_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "rta_internal.h"), os.path.join(CSRC, "rta_device.cuh"),
                  os.path.join(ROOT, "include", "rta.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
]


def stale() -> bool:
    return any(not os.path.exists(lib)
               or any(os.path.getmtime(lib) < os.path.getmtime(d) for d in DEPS)
               for lib in (LIB, TEST_LIB))


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        # one nvcc per translation unit, side by side, then one link
        tag = ".tmp%d" % os.getpid()
        extra = (["-Xptxas", "-v"] if verbose else []) + shlex.split(os.environ.get("RTA_NVCC_EXTRA", ""))
        objs = [os.path.join(HERE, os.path.basename(s)[:-3] + tag + ".o") for s in SOURCES]
        api_testing = os.path.join(HERE, "rta_api_testing" + tag + ".o")
        procs = [subprocess.Popen(["nvcc"] + NVCC_FLAGS + extra + ["-c", "-o", o, s])
                 for s, o in zip(SOURCES, objs)]
        procs.append(subprocess.Popen(["nvcc"] + NVCC_FLAGS + extra + ["-DRTA_TESTING", "-c", "-o",
                                                                      api_testing, SOURCES[-1]]))
        try:
            codes = [p.wait() for p in procs]
            if any(codes):
                raise subprocess.CalledProcessError(max(codes), "nvcc -c")
            for lib, members in ((LIB, objs), (TEST_LIB, objs[:-1] + [api_testing])):
                tmp = lib + tag
                subprocess.check_call(["nvcc"] + NVCC_FLAGS + ["-shared", "-o", tmp] + members)
                os.replace(tmp, lib)
        finally:
            for o in objs + [api_testing]:
                if os.path.exists(o):
                    os.remove(o)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
