"""Static checks of the shipped libvr.so (no GPU needed): what the SASS of every kernel contains and what it does
not.  After a round lost to unexplained "illegal instruction" faults of an asynchronous-copy experiment (DESIGN.md
§10), the product holds no TMA, no mbarrier, no cp.async and no inter-CTA waiting; every kernel is plain loads,
stores, shuffles, CTA barriers and atomics, whose addresses the host emulation (tests/simt) checks against guard
pages.  These tests keep it that way and pin the resources that decide occupancy."""
import re
import subprocess

import pytest

import paper_1111_6661_b200 as vr


@pytest.fixture(scope="module")
def sass():
    vr.load()
    out = subprocess.run(["cuobjdump", "-sass", vr.library_path()], capture_output=True, text=True, check=True).stdout
    kernels, name = {}, None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip()
            kernels[name] = []
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\w+\s+)?([A-Z][A-Z0-9_]*)((?:\.[A-Z0-9_]+)*)", line)
        if m and name:
            kernels[name].append(m.group(1) + m.group(2))
    return kernels


@pytest.fixture(scope="module")
def resources():
    out = subprocess.run(["cuobjdump", "-res-usage", vr.library_path()], capture_output=True, text=True, check=True).stdout
    res, name = {}, None
    for line in out.splitlines():
        m = re.search(r"Function (\S+):", line)
        if m:
            name = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip()
            continue
        m = re.search(r"REG:(\d+) STACK:(\d+) SHARED:(\d+) LOCAL:(\d+)", line)
        if m and name:
            res[name] = tuple(int(x) for x in m.groups())
    return res


def test_no_async_proxy_no_waiting_between_ctas(sass):
    assert len(sass) >= 60
    banned = ("UTMALDG", "UTMASTG", "UBLKCP", "UTMAPF", "SYNCS", "LDGSTS", "NANOSLEEP", "UTC", "LDTM", "STTM",
              "ACQBULK", "CCTL")           # TMA, mbarrier, cp.async, sleeps in spin loops, tcgen05, cluster fences
    for k, ops in sass.items():
        for op in ops:
            assert not op.startswith(banned), (k, op)


def test_no_local_memory_no_stack(sass, resources):
    for k, ops in sass.items():
        assert not [op for op in ops if op.startswith(("LDL", "STL"))], k
    assert len(resources) == len(sass)
    for k, (reg, stack, shared, local) in resources.items():
        assert stack == 0 and local == 0, (k, stack, local)


def test_ray_caster_resources(sass, resources):
    """k_rows: 256 threads per CTA; <= 48 registers keeps 5 CTAs (40 warps) per SM, <= 40 keeps 6 (48 warps); the
    transfer function is the only shared memory; 8 corner loads per sample (+ 1 byte of the skipping grid); packed
    FFMA2 lerps."""
    rows = {k: v for k, v in resources.items() if "k_rows<" in k}
    assert len(rows) == 48                                            # MIP 4 + EA 8 + EA skip 8 + partials 8 + 16-byte loads 12 + 8 (partials)
    for k, (reg, stack, shared, local) in rows.items():
        partials_with_quads = k.split(">(")[0].endswith("true, true")          # the one variant above 48: 4 CTAs per SM
        assert reg <= (64 if partials_with_quads else 48) and shared <= 5200, (k, reg, shared)
    for k, ops in sass.items():
        if "k_rows<" not in k:
            continue
        ldg = [op for op in ops if op.startswith("LDG")]
        args = re.search(r"k_rows<(\d), (\w+), (\w+), (\d), (\w+), (\w+), (\w+)>", k)
        assert args, k
        mode, ert, wide, fast, skip, part, quad = (int(x) if x.isdigit() else x == "true" for x in args.groups())
        n_corner = len([op for op in ldg if ".U8" not in op and ".128" not in op and ".64" not in op])
        if part:                                                      # + the brick table reads of the two fragment flushes
            assert (4 if quad else 8) <= n_corner <= 24, (k, ldg)
        elif quad:                                                    # 4 quads + 4 predicated scalars (+ the staged table)
            assert n_corner == 4 and len([op for op in ldg if ".128" in op]) >= 4, (k, ldg)
        else:
            assert n_corner == 8, (k, ldg)
        assert (len([op for op in ldg if ".U8" in op]) >= 1) == bool(skip), (k, ldg)
        assert len([op for op in ops if op.startswith("FFMA2")]) >= (6 if mode == 1 else 10), k   # 6 paired lerp halves of C.3 (+ C.4, C.5)


def test_reductions_keep_two_ctas_per_sm(resources):
    for k, (reg, stack, shared, local) in resources.items():
        if "k_reduce_" in k or "k_stat" in k and ("_flat" in k or "_box" in k):
            assert reg <= 64, (k, reg)                                # 2 CTAs x 512 threads x 64 registers = the register file
