"""The C-ABI library loads and exports every symbol include/vr.h declares (no GPU needed);
struct layouts in the binding match the header; compute calls fail loudly without a device."""
import ctypes as C
import os
import re
import subprocess

import pytest

import paper_1111_6661_b200 as vr
from paper_1111_6661_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "vr.h")


def declared_functions():
    src = open(HEADER).read()
    return sorted(set(re.findall(r"VR_API\s+[\w\s\*]+?\b(vr_\w+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for n in ("vr_create_volume", "vr_set_transfer_function", "vr_render", "vr_minmax_histogram", "vr_statistics",
              "vr_encode_rgba8"):
        assert n in names
    assert sorted(binding.EXPORTS) == names


def test_library_exports_every_declared_symbol():
    lib = vr.load()
    for n in declared_functions():
        assert hasattr(lib, n), n
    out = subprocess.run(["nm", "-D", "--defined-only", vr.library_path()], capture_output=True, text=True).stdout
    exported = {l.split()[-1] for l in out.splitlines() if " T " in l}
    assert set(declared_functions()) <= exported
    assert not [s for s in exported if s.startswith("oracle_")]          # shares nothing with the oracle
    assert "sm_100a" in vr.vr_version()


def test_library_is_built_for_sm_100a_only():
    out = subprocess.run(["cuobjdump", "--list-elf", vr.library_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, out


def test_struct_sizes_match_header(tmp_path):
    src = tmp_path / "sz.c"
    src.write_text('#include "vr.h"\n#include <stdio.h>\n#include <stddef.h>\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu %zu\\n",'
                   "sizeof(vr_volume_desc),sizeof(vr_camera),sizeof(vr_image),sizeof(vr_stats),"
                   "offsetof(vr_summary,counts),offsetof(vr_volume_desc,data),sizeof(vr_statistics_result),"
                   "offsetof(vr_statistics_result,median));return 0;}\n")
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True).stdout.split()]
    assert got[0] == C.sizeof(binding.vr_volume_desc)
    assert got[1] == C.sizeof(binding.vr_camera)
    assert got[2] == C.sizeof(binding.vr_image)
    assert got[3] == C.sizeof(binding.vr_stats)
    assert got[4] == 32 and binding.summary_dtype(256).itemsize == 32 + 8 * 256
    assert got[5] == binding.vr_volume_desc.data.offset
    assert got[6] == C.sizeof(binding.vr_statistics_result) == binding.STATISTICS_DTYPE.itemsize == 40
    assert got[7] == binding.vr_statistics_result.median.offset == 32


def test_argument_errors_without_gpu():
    lib = vr.load()
    h = C.c_void_p()
    assert lib.vr_create_volume(None, C.byref(h)) == vr.VR_ERR_INVALID_ARG
    assert b"NULL" in lib.vr_last_error()
    d = binding.vr_volume_desc()
    d.struct_size = 3
    assert lib.vr_create_volume(C.byref(d), C.byref(h)) == vr.VR_ERR_INVALID_ARG
    d.struct_size = C.sizeof(d)
    d.nx, d.ny, d.nz = 1, 8, 8
    assert lib.vr_create_volume(C.byref(d), C.byref(h)) == vr.VR_ERR_INVALID_ARG
    assert lib.vr_render(None, None, 0, None, None) == vr.VR_ERR_INVALID_ARG
    assert lib.vr_minmax_histogram(None, 256, None, None, 0, None) == vr.VR_ERR_INVALID_ARG
    assert lib.vr_destroy_volume(None) == vr.VR_OK


def test_no_cpu_fallback_without_device():
    """Without a CUDA device a well-formed create call must fail with VR_ERR_CUDA, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import numpy as np
    buf = np.zeros(8 * 8 * 8 + 4, dtype=np.float32)
    addr = (buf.ctypes.data + 15) & ~15
    d = binding.vr_volume_desc()
    d.struct_size = C.sizeof(d)
    d.nx = d.ny = d.nz = 8
    d.data = addr
    h = C.c_void_p()
    rc = vr.load().vr_create_volume(C.byref(d), C.byref(h))
    assert rc == vr.VR_ERR_CUDA and not h.value
    assert b"CUDA error" in vr.load().vr_last_error()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1111_6661_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower().replace("no cpu fallback", ""), f


def test_c_client_compiles_and_links_against_the_library(tmp_path):
    """A plain C translation unit that uses every entry point of include/vr.h the way README.md shows compiles with
    -Wall -Werror and links against libvr.so (C linkage, no CUDA or C++ types in the interface); it is not run."""
    src = tmp_path / "client.c"
    src.write_text(r'''
#include "vr.h"
#include <stddef.h>
int client(const float *dev_voxels, float *dev_img, vr_summary *sum_dev, unsigned char *frame, void *stream,
           const float *tf, vr_statistics_result *st)
{
    vr_volume_desc d = { sizeof d, 64, 64, 64, 16, VR_LINEAR, VR_DEVICE, 0, dev_voxels, 0 };
    vr_volume *vol = NULL;
    if (vr_create_volume(&d, &vol) != VR_OK) return 1;
    vr_minmax_histogram(vol, 256, NULL, sum_dev, VR_DEVICE, stream);
    vr_set_transfer_function(vol, tf, -1.0f, 1.0f);
    vr_camera cam = { sizeof cam, 32, 32, {0, 0, -1}, {2, 0, 0}, {0, 2, 0}, {0, 0, 1}, {0, 0, 0}, {0, 0, 0}, 1.0f, 0.99f, 0 };
    vr_image img = { sizeof img, 4, VR_DEVICE, 0, dev_img, 0 };
    vr_render(vol, &cam, VR_EA, &img, stream);
    vr_encode_desc e = { sizeof e, 32, 32, VR_EA, {0, 0, 0}, 0, 0 };
    vr_encode_rgba8(vol, &e, &img, frame, 0, VR_HOST_PINNED, stream);
    vr_statistics(vol, st, VR_HOST_PINNED, stream);
    vr_set_option(vol, VR_OPT_EMPTY_SKIP, 1);
    vr_stats s = { sizeof s };
    vr_get_stats(vol, &s);
    return vr_destroy_volume(vol) == VR_OK && vr_last_error()[0] == 0 && vr_version() != NULL ? 0 : 2;
}
int main(void) { return 0; }
''')
    exe = tmp_path / "client"
    lib = vr.library_path()
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-Wno-missing-field-initializers", "-I", os.path.join(ROOT, "include"),
                    str(src), "-o", str(exe), "-L", os.path.dirname(lib), "-l:" + os.path.basename(lib),
                    "-Wl,-rpath," + os.path.dirname(lib)], check=True)
