"""Static resources of the default ray-cast kernel, from `nvcc -Xptxas -v` (no GPU needed): k_shear must not spill
and must stay within 85 registers per thread, or three 256-thread CTAs no longer fit an SM (65536 registers) and the
host plan's occupancy assumptions break silently."""
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_k_shear_registers_and_spills(tmp_path):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    src = os.path.join(ROOT, "paper_1111_6661_b200", "csrc", "vr_shear.cu")
    r = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "--fmad=false",
                        "-Xptxas", "-v", "-c", src, "-o", str(tmp_path / "vr_shear.o")], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    out = r.stdout + r.stderr
    blocks = [b for b in out.split("Compiling entry function")[1:] if "k_shear" in b.splitlines()[0]]
    assert len(blocks) == 3, out                          # MIP, EA, EA + ERT
    for b in blocks:
        regs = int(re.search(r"Used (\d+) registers", b).group(1))
        assert regs <= 85, b
        assert "0 bytes spill stores, 0 bytes spill loads" in b, b
