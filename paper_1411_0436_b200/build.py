"""Build step: nvcc -> paper_1411_0436_b200/libspec.so (in-tree, sm_100a only).

`python -m paper_1411_0436_b200.build [--force]`.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libspec.so")
SOURCES = [os.path.join(CSRC, "spec.cu")]
DEPS = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh", ".h"))] + [
    os.path.join(_ROOT, "include", "spec.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
    # NO "-split-compile": the parallel split is a race.  The same command line produced one of two code generations
    # of the same source from run to run (measured on one B200, profiles/r02_experiments.md row 24: 117 or 110 GHz at
    # configs[1], 146 or 138 GHz at direct FFT 32768, and the other way round 266 or 282 GHz at direct FFT 4096).
    # Without it the build takes four minutes instead of one and a half, and is byte-for-byte reproducible; the source
    # is named relative to csrc/ so that the repository's location does not enter the binary either.
]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        extra = os.environ.get("SPEC_NVCC_EXTRA", "").split()   # e.g. -DSPEC_FUSED_DEBUG_COUNTERS
        cmd = ([nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB]
               + [os.path.relpath(p, CSRC) for p in SOURCES])
        subprocess.check_call(cmd, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
