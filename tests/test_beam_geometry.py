"""Host brute-force check of the beam geometry the sheared-plane kernel stages by (vr_beamgeom.cuh): no voxel a
sample of a beam can read may lie outside plane_rect() of the data plane it is read from, and no plane between two
planes of a beam may need a larger rectangle than beam_rect_bound() plus one (the kernel's fit test); a host model of
the kernel's step loop, running the kernel's own schedule functions, checks that every base plane is marched once, in
order, from resident ring slots that no in-flight copy can overwrite.  Compiles
tests/geom_check.cu as HOST code with nvcc (no GPU needed) and runs it."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_plane_rect_contains_every_sample_footprint(tmp_path):
    exe = str(tmp_path / "geom_check")
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-O2", "-std=c++17", "-o", exe, os.path.join(ROOT, "tests", "geom_check.cu")], check=True,
                   capture_output=True)
    r = subprocess.run([exe, "120"], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rect_bad 0" in r.stdout and "convex_bad 0" in r.stdout and "schedule_bad 0" in r.stdout
