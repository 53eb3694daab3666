"""Build the CUDA library in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(CSRC, "libeldr_moe.so")
SOURCES = ["eldr_moe.cu"]


def _headers():
    """Every header the translation unit can include: a change to any of them rebuilds the library."""
    import glob
    return sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")))


def _stale(lib: str = None) -> bool:
    lib = lib or LIB
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in SOURCES] + _headers() + [os.path.join(_ROOT, "include", "eldr_moe.h")]
    return any(os.path.getmtime(d) > t for d in deps)


TRACE_LIB = os.path.join(CSRC, "libeldr_moe_trace.so")


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    """trace=True builds a SECOND library, libeldr_moe_trace.so, with -DELDR_TRACE: the fused kernel then stamps
    %globaltimer at its milestones (`bench.py --timeline`).  The measured library carries no trace code."""
    lib = TRACE_LIB if trace else LIB
    if not force and not _stale(lib):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(_ROOT, "include"), "-I", CSRC,
           "-o", lib] + [os.path.join(CSRC, s) for s in SOURCES]
    cmd[1:1] = os.environ.get("ELDR_EXTRA_NVCC_FLAGS", "").split() + (["-DELDR_TRACE"] if trace else [])
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
