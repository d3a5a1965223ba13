"""CPU oracle — TEST INFRASTRUCTURE ONLY (see vr_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_1111_6661_b200 and shares no code with it.
"""
from .oracle import (build, render, minmax_hist, statistics, encode_rgba8, num_threads, RenderResult, Summary, Statistics,
                     EA, MIP, F32, F64, LINEAR, BRICKED_HALO1)

__all__ = ["build", "render", "minmax_hist", "statistics", "encode_rgba8", "num_threads", "RenderResult", "Summary", "Statistics",
           "EA", "MIP", "F32", "F64", "LINEAR", "BRICKED_HALO1"]
