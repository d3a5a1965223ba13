"""The HOST plan of the sheared-plane kernel on the real configs, without a GPU: tests/shear_plan_check.cu includes
vr_shear.cu, runs make_shear_plan() on cameras written here from workload/, and replays per beam the fit decision of
the kernel prologue and the planner's per-plane check with the same geometry functions.  On cfg1, cfg2 (orbit) and
cfg4 (3840x2160, 64 GiB dims) no beam may fall back to global memory (a slow tail), no plane may overflow its slot,
and the plan must keep its invariants (ring >= 2G+1 slots, shared memory within the CTA limit)."""
import os
import re
import subprocess

import workload as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _line(cfg, view):
    cam = cfg.camera(view)
    v = cam.vectors().ravel()
    return "%d %d %d %d %d %r " % (*cfg.dims, cam.width, cam.height, float(cam.step)) + " ".join("%.9g" % x for x in v)


def test_plan_has_no_fallback_beams_on_the_configs(tmp_path):
    exe, cams = str(tmp_path / "shear_plan_check"), str(tmp_path / "cams.txt")
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-arch=sm_100a", "-O2", "-std=c++17", "-o", exe, os.path.join(ROOT, "tests", "shear_plan_check.cu")],
                   check=True, capture_output=True)
    with open(cams, "w") as f:
        f.write(_line(W.get_config(1), 0) + "\n")
        for view in (0, 1, 2, 3, 6, 13):
            f.write(_line(W.get_config(2), view) + "\n")
        for view in (0, 12):
            f.write(_line(W.get_config(4), view) + "\n")
    r = subprocess.run([exe, cams], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    assert re.search(r"total beams \d+ direct_fit 0 overflow 0", r.stdout), r.stdout
    # cfg2 keeps three CTAs per SM on every view; cfg4 (sparse sampling, 70x70-voxel planes) at least two
    ctas = [int(m) for m in re.findall(r" ctas (\d)", r.stdout)]
    assert all(c == 3 for c in ctas[:7]) and all(c >= 2 for c in ctas[7:]), r.stdout
