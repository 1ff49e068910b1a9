"""In-tree build of libwl.so (the CUDA library behind include/wl.h) for sm_100a with plain nvcc.

``python -m paper_2304_08159_b200.build`` or ``build_cuda()``.  nvcc cross-compiles without a GPU.  The CUDA runtime
is linked statically, so the .so needs nothing but the NVIDIA driver at run time.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libwl.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
    # No FMA contraction: every multiply and add rounds separately, exactly as the oracle's (-ffp-contract=off), which
    # makes the fp32 and fp64 iterates and residual histories bit-identical to it (DESIGN.md §3 reading 12; measured
    # cost: 5 % of the 512^3 V-cycle).  Explicit fmaf() calls (the reciprocal's Newton steps) stay fused.
    "-fmad=false",
]


def _sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    inc = os.path.join(os.path.dirname(HERE), "include", "wl.h")
    return _sources() + sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h"))) + [inc]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _deps())


def build_cuda(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = LIB + f".tmp{os.getpid()}"
    extra = os.environ.get("WL_NVCC_EXTRA", "").split()   # A/B builds, e.g. WL_NVCC_EXTRA=-DWL_FP64_C_PLANE=1
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + _sources()
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if verbose:
        sys.stderr.write(res.stdout + res.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_cuda(force="--force" in sys.argv, verbose="-v" in sys.argv))
