#!/usr/bin/env python
"""Writes tests/golden/oracle_tiny.txt: bit patterns of what the CPU oracle computes on one tiny seeded case.

The paper (arxiv/paper_1111_6661) prints no worked example, so this is NOT a pin of the oracle against the
paper (those are the closed-form pins of tests/test_oracle_pins.py); it is a regression guard: a later change
to the oracle's arithmetic must change this file in the same commit and say why.  Calls only
oracle/ and workload/ — never the CUDA path.

    python tests/golden/make_oracle_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle as O  # noqa: E402
import workload as W  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny.txt")


def case():
    n = (12, 10, 14)
    v = W.make_cube(W.Recipe(*n, seed=0x1111666100000001, n_sources=2))
    cam = W.perspective_camera((31.5, 17.25, -22.0), (6, 5, 7), (0, 1, 0), 38.0, 6, 5, step=0.5, ert_alpha=0.99)
    s = O.minmax_hist(v, 16)
    tf = W.tf_opaque(n, 0.5)
    ea = O.render(v, cam, O.EA, tf, s.vmin, s.vmax)
    mip = O.render(v, cam, O.MIP)
    eab = O.render(v, cam.with_(ert_alpha=0.0), O.EA, tf, s.vmin, s.vmax, brick=4)
    st = O.statistics(v)
    frame = O.encode_rgba8(ea.image, O.EA, background=(0.1, 0.2, 0.3))
    return v, s, ea, mip, eab, st, frame


def lines():
    v, s, ea, mip, eab, st, frame = case()
    yield "# written by tests/golden/make_oracle_golden.py (oracle only); float32 bit patterns in hex"
    yield "cube_checksum %016x" % W.checksum(v)
    yield "minmax %08x %08x" % (np.float32(s.vmin).view(np.uint32), np.float32(s.vmax).view(np.uint32))
    yield "hist16 " + " ".join(str(int(c)) for c in s.counts)
    yield "K " + " ".join(str(int(k)) for k in ea.K.ravel())
    yield "K_ert " + " ".join(str(int(k)) for k in ea.K_ert.ravel())
    yield "ea_ert " + " ".join("%08x" % x for x in ea.image.view(np.uint32).ravel())
    yield "mip " + " ".join("%08x" % x for x in mip.image.view(np.uint32).ravel())
    yield "ea_bricked4 " + " ".join("%08x" % x for x in eab.image.view(np.uint32).ravel())
    yield "statistics %d %d %016x %016x %08x" % (st.n_finite, st.n_nonfinite, np.float64(st.mean).view(np.uint64),
                                                 np.float64(st.stddev).view(np.uint64), np.float32(st.median).view(np.uint32))
    yield "frame_rgba8 " + " ".join("%02x" % x for x in frame.ravel())


if __name__ == "__main__":
    with open(OUT, "w") as f:
        f.write("\n".join(lines()) + "\n")
    print("wrote", OUT)
