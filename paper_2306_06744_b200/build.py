"""Build step: compile csrc/*.cu into paper_2306_06744_b200/liblt.so for sm_100a.

    python -m paper_2306_06744_b200.build [--force]

nvcc cross-compiles without a GPU.  The shared library is built in-tree (git-ignored) so it
travels to the GPU box with the snapshot.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblt.so")
LIB_DEBUG = os.path.join(HERE, "liblt_debug.so")  # -DLT_DEBUG: device-side bounds / protocol assertions
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC", "-cudart", "static", "--threads", "0",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale(lib=LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(INCLUDE, "*.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, debug: bool = False) -> str:
    """debug=True: the checked build liblt_debug.so (-DLT_DEBUG; load it with LT_DEBUG_LIB=1)."""
    lib = LIB_DEBUG if debug else LIB
    if not force and not _stale(lib):
        return lib
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = lib + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-DLT_DEBUG"] if debug else []) + (["-Xptxas", "-v"] if verbose else []) + \
        ["-o", tmp] + sources()
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug="--debug" in sys.argv))
