"""TEST INFRASTRUCTURE: builds tests/simt/libvr_simt.so — the library's own sources (csrc/*.cu: host runtime AND
kernels) compiled by g++ against tests/simt/simt_host.h, which executes every CUDA thread as a fiber on the host
(see that header).  Used only by tests/test_simt_parity.py; the product (paper_1111_6661_b200/libvr.so, nvcc,
sm_100a) never loads it."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_1111_6661_b200", "csrc")
UBSAN = bool(os.environ.get("VR_SIMT_UBSAN"))
LIB = os.path.join(HERE, "libvr_simt_ubsan.so" if UBSAN else "libvr_simt.so")


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cu"))


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, f) for f in os.listdir(HERE) if not f.endswith(".so")]
    deps.append(os.path.join(ROOT, "include", "vr.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False) -> str:
    if force or stale():
        objs = []
        flags = ["-std=c++17", "-O2", "-g", "-fPIC", "-fvisibility=hidden", "-mfma", "-ffp-contract=off",
                 "-fno-strict-aliasing", "-Wall", "-Wno-unknown-pragmas", "-Wno-unused-function"]
        if UBSAN:                                # VR_SIMT_UBSAN=1: abort on out-of-bounds indices of fixed-size (shared-
            flags += ["-fsanitize=bounds,shift,integer-divide-by-zero,signed-integer-overflow,null,alignment",   # memory)
                      "-fno-sanitize-recover=all"]       # arrays, misaligned vector accesses, signed overflow, bad shifts
        cmd = ["g++"] + flags + ["-shared", "-o", LIB]
        for s in sources():
            cmd += ["-x", "c++", "-include", os.path.join(HERE, "simt_host.h"), s]
        cmd += ["-x", "c++", os.path.join(HERE, "simt_runtime.cpp")]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv))
