"""Host brute force of the pixel-to-lane map of the default ray-caster (csrc/vr_lanemap.h and the pixel formula of
k_rows): every pixel is rendered exactly once for any camera, image size, volume copy and pixel class.  Compiles
tests/lanemap_check.cpp with g++ and runs it (no GPU needed)."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_every_pixel_exactly_once(tmp_path):
    exe = str(tmp_path / "lanemap_check")
    subprocess.run(["g++", "-O2", "-std=c++17", "-mfma", "-ffp-contract=off", "-o", exe,
                    os.path.join(ROOT, "tests", "lanemap_check.cpp")], check=True, capture_output=True)
    r = subprocess.run([exe, "240"], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    assert " bad 0" in r.stdout
