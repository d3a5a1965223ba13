"""TEST INFRASTRUCTURE — parity of the library's own kernels at the configs' FULL sizes, in the host emulation.

The emulation (tests/simt) executes the CUDA sources thread by thread at about 3e6 samples per second, which is enough
to render whole frames of cfg2 (1 GiB cube, 1024^2 image, 3.3e8 samples) and cfg3 (8 GiB cube, 1920x1080, 7.3e8
samples, sort-last) and to run the summary and statistics passes over the whole cubes — every output compared bit for
bit with the oracle on the same bytes.  It needs no GPU, tens of GB of host memory and the better part of an hour;
it is not part of the pytest suite.  cfg4 (64 GiB + copies) does not fit this box.

    python tests/simt/full_size_emulated.py [--cfg2-views 0,1,..] [--cfg3-views 1,5] > profiles/r2_full_size_emulated_parity.md
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
sys.path.insert(0, HERE)

import simt_lib  # noqa: E402
import oracle as O  # noqa: E402
import paper_1111_6661_b200 as vr  # noqa: E402
import workload as W  # noqa: E402
from backends import BACKENDS, render, statistics, summary  # noqa: E402


def host_cube(cfg):
    nx, ny, nz = cfg.dims
    out = np.empty((nz, ny, nx), dtype=np.float32)
    gen = W.CubeGenerator(cfg.recipe)
    slab = max(1, (1 << 28) // (nx * ny))
    for z0 in range(0, nz, slab):
        gen.fill(out[z0:min(nz, z0 + slab)], z0, min(nz, z0 + slab))
    return out


def same(a, b):
    return bool(np.array_equal(a, b, equal_nan=True))


def run_config(be, number, views, do_stats):
    cfg = W.get_config(number)
    v = host_cube(cfg)
    tf = W.tf_haze(cfg.dims, cfg.step)
    print(f"\n## cfg{number}: {cfg.dims[0]}x{cfg.dims[1]}x{cfg.dims[2]} ({v.nbytes / 2**30:.0f} GiB), {cfg.width}x{cfg.height}, step {cfg.step}, "
          f"modes {'+'.join(cfg.modes)}, ERT {cfg.ert_alpha}, {'sort-last, ' if cfg.sort_last else ''}bricks {cfg.brick}^3\n")
    print("| what | result | emulated s | oracle s | detail |")
    print("|---|---|---:|---:|---|")
    ok = True
    with be.ctx():
        with vr.Volume(be.dev(v), cfg.dims, brick=cfg.brick) as vol:
            t = time.time(); g = summary(be, vol); te = time.time() - t
            t = time.time(); o = O.minmax_hist(v); to = time.time() - t
            good = g["vmin"] == o.vmin and g["vmax"] == o.vmax and same(g["counts"], o.counts) and int(g["n_nonfinite"]) == o.n_nonfinite
            ok &= good
            print(f"| vr_minmax_histogram (256 bins, whole cube) | {'bit-exact' if good else 'DIFFERS'} | {te:.0f} | {to:.0f} | "
                  f"vmin {float(o.vmin):.6g} vmax {float(o.vmax):.6g} |", flush=True)
            if do_stats:
                t = time.time(); s = statistics(be, vol); te = time.time() - t
                t = time.time(); so = O.statistics(v); to = time.time() - t
                scale = float(np.abs(v).mean())
                good = (int(s["n_finite"]) == so.n_finite and np.float32(s["median"]).tobytes() == np.float32(so.median).tobytes()
                        and abs(float(s["mean"]) - so.mean) <= 1e-13 * scale and abs(float(s["stddev"]) - so.stddev) <= 1e-13 * max(so.stddev, scale))
                ok &= good
                print(f"| vr_statistics (whole cube) | {'median bit-exact, moments within 1e-13' if good else 'DIFFERS'} | {te:.0f} | {to:.0f} | "
                      f"mean {so.mean:.12g} stddev {so.stddev:.12g} median {float(so.median):.9g} |", flush=True)
            vol.set_transfer_function(tf, float(o.vmin), float(o.vmax))
            for view in views:
                cam = cfg.camera(view)
                for mode in cfg.modes:
                    m = vr.VR_EA if mode == "ea" else vr.VR_MIP
                    t = time.time(); gi = render(be, vol, cam, m); te = time.time() - t
                    st = vol.stats()
                    t = time.time()
                    oi = O.render(v, cam, O.EA if mode == "ea" else O.MIP, tf, float(o.vmin), float(o.vmax),
                                  brick=cfg.brick if cfg.sort_last else 0)
                    to = time.time() - t
                    good = same(gi, oi.image)
                    ok &= good
                    print(f"| view {view} {mode.upper()} | {'bit-identical' if good else 'DIFFERS'} | {te:.0f} | {to:.0f} | "
                          f"{oi.n_nominal} nominal samples, path {st['path']}, launches {st['kernel_launches']}, with 16-byte loads "
                          f"{st['quad_launches']}, z-fastest copy {st['zfast_copy']}, fragments {st['fragments']} |", flush=True)
    del v
    return ok


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg2-views", default=",".join(str(i) for i in range(16)))
    ap.add_argument("--cfg3-views", default="1,5")
    args = ap.parse_args()
    simt_lib.lib().simt_set_device_capacity(40 << 30)
    be = BACKENDS["simt"]
    print("# r2 — parity at the configs' full sizes, library kernels executed in the host emulation\n")
    print(f"Command: `python tests/simt/full_size_emulated.py --cfg2-views {args.cfg2_views} --cfg3-views {args.cfg3_views}` (no GPU; "
          "the CUDA sources of libvr compiled by g++ against tests/simt and executed thread by thread; outputs compared with the "
          "oracle on the same bytes).  This is what `pytest -m gpu` checks on a B200 (`test_cfg2_full_size_sampled`, "
          "`test_cfg3_full_size_sampled`), here on EVERY pixel instead of a lattice.")
    ok = True
    if args.cfg2_views:
        ok &= run_config(be, 2, [int(x) for x in args.cfg2_views.split(",")], True)
    if args.cfg3_views:
        ok &= run_config(be, 3, [int(x) for x in args.cfg3_views.split(",")], False)
    print("\n**" + ("ALL BIT-IDENTICAL" if ok else "DIFFERENCES FOUND") + "**")
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
