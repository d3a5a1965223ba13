"""Host brute-force check of the per-frame brick plan (vr_plan.h, used by plan_bricks() of vr_api.cu): screen
rectangles contain every pixel whose ray owns a sample in the brick, and owner bricks appear in ascending visibility
key along every ray (C.7), for perspective (also eye inside the volume) and orthographic cameras.  Compiles
tests/plan_check.cpp with g++ and runs it (no GPU needed)."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_brick_rectangles_and_visibility_order(tmp_path):
    exe = str(tmp_path / "plan_check")
    subprocess.run(["g++", "-O2", "-std=c++17", "-mfma", "-ffp-contract=off", "-o", exe, os.path.join(ROOT, "tests", "plan_check.cpp")], check=True,
                   capture_output=True)
    r = subprocess.run([exe, "80"], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rect_bad 0" in r.stdout and "order_bad 0" in r.stdout
    # the same at the sizes, brick edges, images and orbit cameras of cfg3 / cfg4 / cfg5, with float32 rays (C.1-C.3)
    r = subprocess.run([exe, "0", "configs"], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rect_bad 0" in r.stdout and "order_bad 0" in r.stdout
