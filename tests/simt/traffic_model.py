"""TEST INFRASTRUCTURE — memory-traffic model of the ray-caster's corner loads, measured in the host emulation
(tests/simt): the library's own kernels run thread by thread on scaled-down copies of the BASELINE.json configs
(same cameras, same pixel-spacing-to-voxel ratio, same step), and for every warp-level load instruction the
emulation counts the distinct 128-byte lines (what the L1 tag stage and the LSU pay per instruction) and the
distinct 32-byte sectors (what L2 / HBM are asked for, before any cache hit) that the ACTIVE lanes touch, and how
many lanes were active (lane efficiency of the lag-synchronised march).  No timing: counts only.

    python tests/simt/traffic_model.py [--configs 2,4] [--views 4] > profiles/r2_lane_traffic_model.md

Writes a markdown table to stdout."""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, HERE)

import simt_lib  # noqa: E402
import paper_1111_6661_b200 as vr  # noqa: E402
import workload as W  # noqa: E402

SCALE = {2: 1 / 8, 3: 1 / 16, 4: 1 / 16}


def run(cfg, v, cam, mode, variant):
    path, zcopy, lag = variant[:3]
    tile = variant[3] if len(variant) > 3 else 1
    lib = simt_lib.lib()
    with simt_lib.emulated():
        d = simt_lib.Buffer.of(v, device=True)
        with vr.Volume(d, cfg.dims) as vol:
            vol.set_option(vr.VR_OPT_RENDER_PATH, path)
            vol.set_option(vr.VR_OPT_ZFAST_COPY, zcopy)
            vol.set_option(vr.VR_OPT_LANE_LAG, lag)
            vol.set_option(vr.VR_OPT_TILE_SHEAR, tile)
            vol.set_option(vr.VR_OPT_EMPTY_SKIP, 0)
            vol.set_option(vr.VR_OPT_ROW_LOADS, 0)                   # the trace counts the scalar loads (+ the quad what-if)
            vol.set_transfer_function(W.tf_haze(cfg.dims, cfg.step), -6.0, 24.0)
            out = simt_lib.Buffer((cam.height, cam.width, 4) if mode == vr.VR_EA else (cam.height, cam.width))
            lib.simt_trace(1)
            vol.render(cam, mode, out=out, stream=0)
            st = [lib.simt_trace_stat(i) for i in range(8)]
            lib.simt_trace(0)
    return st


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="2,3,4")
    ap.add_argument("--views", type=int, default=4)
    args = ap.parse_args()
    variants = [("ray-major 8x4-pixel warps (path 1)", (1, 1, 1)),
                ("lane-mapped, x-fastest array only, lag 1", (0, 0, 1)),
                ("lane-mapped + z-fastest copy, lag 0 (no lane synchronisation)", (0, 1, 0)),
                ("lane-mapped + z-fastest copy, lag 1, one shear per frame", (0, 1, 1, 0)),
                ("lane-mapped + z-fastest copy, lag 1 (default)", (0, 1, 1)),
                ("lane-mapped + z-fastest copy, lag 4", (0, 1, 4))]
    print("# Memory-traffic model of the corner loads (host emulation of the library's kernels)\n")
    print("Command: `python tests/simt/traffic_model.py --configs %s --views %d` (no GPU; counts, not times).\n" % (args.configs, args.views))
    print("Per warp-level load instruction (8 per sample): distinct 128-byte lines and 32-byte sectors touched by the active "
          "lanes; lane efficiency = active lanes / (32 x warp iterations).  A fully coalesced load of 32 active lanes reads "
          "1-2 lines and 4-5 sectors.  Configs are scaled copies (volume and image by the same factor, so the pixel "
          "spacing in voxels — what decides coalescing — is the config's own).\n")
    print("`lines / sample` = 8 loads x lines per load / active lanes: the L1 cost of one sample.  `what-if 16 B` = the same with "
          "ONE aligned 16-byte load per row (+ a scalar load for the lanes whose x is the last element of its quad) instead of "
          "two scalar loads: what `k_rows<QUAD>` (VR_OPT_ROW_LOADS) does, counted from the scalar trace.  `samples that load`: "
          "with a step below one voxel a ray keeps the 8 voxels of its cell in registers, and a sample in the same cell as the ray's "
          "previous one loads nothing (lane-mapped kernel only).\n")
    print("| config (scale) | view | variant | samples | lane efficiency | lines / load | sectors / load | lines / sample | what-if 16 B: lines / sample | samples that load |")
    print("|---|---|---|---:|---:|---:|---:|---:|---:|---:|")
    for number in (int(x) for x in args.configs.split(",")):
        cfg = W.get_config(number, scale=SCALE[number])
        v = W.make_cube(cfg.recipe)
        mode = vr.VR_EA if "ea" in cfg.modes else vr.VR_MIP
        views = list(range(0, cfg.n_views, max(1, cfg.n_views // args.views)))[: args.views]
        totals = {name: np.zeros(8) for name, _ in variants}
        for view in views:
            cam = cfg.camera(view).with_(flags=0)
            for name, var in variants:
                st = np.array(run(cfg, v, cam, mode, var), dtype=np.float64)
                totals[name] += st
                it, act, ld, ln, sc, qld, qln, nld = st
                print(f"| cfg{number} ({SCALE[number]:g}) | {view} | {name} | {int(act)} | {act / (32 * it):.2f} | {ln / ld:.2f} | "
                      f"{sc / ld:.2f} | {ln / act:.2f} | {qln / act:.2f} | {nld / act:.2f} |")
        for name, _ in variants:
            it, act, ld, ln, sc, qld, qln, nld = totals[name]
            print(f"| **cfg{number} all views** | | **{name}** | {int(act)} | **{act / (32 * it):.2f}** | **{ln / ld:.2f}** | "
                  f"**{sc / ld:.2f}** | **{ln / act:.2f}** | **{qln / act:.2f}** | {nld / act:.2f} |")


if __name__ == "__main__":
    main()
