"""Build libvr.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvr.so")
SOURCES = ["vr_api.cu", "vr_reduce.cu", "vr_stats.cu", "vr_raycast.cu", "vr_lanes.cu", "vr_macro.cu", "vr_encode.cu"]
HEADERS = ["vr_internal.h", "vr_plan.h", "vr_math.cuh", "vr_range.cuh", "vr_sweep.cuh", "vr_lanemap.h", os.path.join("..", "..", "include", "vr.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--fmad=false",                 # nothing is contracted behind the canonical arithmetic's back
    "-Xcompiler", "-fPIC,-fvisibility=hidden,-O2,-mfma,-ffp-contract=off",   # fmaf inlined in the host plans, nothing contracted implicitly
    "-shared", "-cudart", "static",
]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
