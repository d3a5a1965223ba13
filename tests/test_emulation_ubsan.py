"""A subset of the emulated parity tests once more with the library's CUDA sources compiled under UBSan
(-fsanitize=bounds,alignment,signed-integer-overflow,shift,null,integer-divide-by-zero, no recovery): an index past
the end of a fixed-size shared-memory array, a misaligned 16-byte vector access (ld_stream4, the QUAD row loads,
float4 image stores) or an overflowing offset computation aborts the run.  Global-memory bounds are the guard pages'
job (simt_runtime.cpp)."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_emulated_parity_subset_under_ubsan():
    env = dict(os.environ, VR_SIMT_UBSAN="1")
    sel = "cfg1 or 16_byte or statistics_special or statistics_bricked or leaps_over or minmax_hist_nonfinite or " \
          "(sort_last_equals and 16) or 64_bit or empty_bricks or degenerate"
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_parity.py"), "-x", "-q",
                        "-m", "not gpu", "-k", sel, "-p", "no:cacheprovider"], env=env, capture_output=True, text=True,
                       cwd=ROOT, timeout=1500)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "runtime error" not in r.stderr and " passed" in r.stdout
