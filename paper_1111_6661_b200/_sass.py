"""Static report of the built libvr.so (no GPU needed): registers / shared memory / occupancy of every kernel and the
SASS of the innermost loop of the ray-caster variants the benchmark configs launch.

    python -m paper_1111_6661_b200._sass > profiles/r2_sass_k_rows.md
"""
from __future__ import annotations

import re
import subprocess

from . import _build


def _demangle(name: str) -> str:
    return subprocess.run(["c++filt", name], capture_output=True, text=True).stdout.strip()


def kernels():
    lib = _build.build()
    res = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    usage, name = {}, None
    for line in res.splitlines():
        m = re.search(r"Function (\S+):", line)
        if m:
            name = _demangle(m.group(1))
            continue
        m = re.search(r"REG:(\d+) STACK:(\d+) SHARED:(\d+) LOCAL:(\d+)", line)
        if m and name:
            usage[name] = tuple(int(x) for x in m.groups())
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    code, name = {}, None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = _demangle(m.group(1))
            code[name] = []
            continue
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m and name:
            code[name].append((int(m.group(1), 16), m.group(2).strip()))
    return usage, code


def inner_loop(ins):
    """The longest backward-branch region that contains a global load."""
    best = []
    for addr, txt in ins:
        m = re.search(r"BRA\s+(?:!?U?P\d+,\s*)?0x([0-9a-f]+)", txt)
        if m and int(m.group(1), 16) < addr:
            tgt = int(m.group(1), 16)
            body = [(a, t) for a, t in ins if tgt <= a <= addr]
            if any("LDG" in t for _, t in body) and len(body) > len(best):
                best = body
    return best


def short(name: str) -> str:
    return re.sub(r"\(.*$", "", name.replace("vr::(anonymous namespace)::", "").replace("void ", ""))


def main():
    usage, code = kernels()
    print("# r2 — static SASS report of libvr.so (sm_100a only)\n")
    print("Command: `python -m paper_1111_6661_b200._sass` (cuobjdump -res-usage / -sass of the in-tree build; no GPU).  nvcc "
          "12.9, `-gencode arch=compute_100a,code=sm_100a -O3 --fmad=false -lineinfo`.\n")
    print("## Every kernel\n")
    print("| kernel | registers | static shared B | threads / CTA | CTAs / SM by registers |")
    print("|---|---:|---:|---:|---:|")
    for k in sorted(usage):
        reg, stack, shared, local = usage[k]
        thr = 256 if ("k_rows" in k or "k_macro" in k or "k_encode" in k or "k_transpose" in k or "k_composite" in k
                      or "k_fragment" in k or "k_brick" in k or "k_chain_init" in k or "k_chain_finish" in k) else \
            512 if ("k_reduce" in k or "k_stat0" in k or "k_stat_sel" in k) else 128 if ("k_march" in k or "k_chain_brick" in k) else 1
        per_sm = min(2048 // max(thr, 32), 65536 // (max(reg, 16) * thr)) if thr > 1 else "-"
        print(f"| `{short(k)}` | {reg} | {shared} | {thr} | {per_sm} |")
    assert all(u[1] == 0 and u[3] == 0 for u in usage.values())
    print("\nNo kernel uses a stack or local memory.  Opcodes that never occur: UTMALDG / UBLKCP (TMA), SYNCS (mbarrier), "
          "LDGSTS (cp.async), UTC*MMA / LDTM (tcgen05), NANOSLEEP (`tests/test_kernel_static.py`).\n")
    print("## Sample loop of the ray-caster (`k_rows<MODE, ERT, WIDE, FAST, SKIP, PART, QUAD>`)\n")
    print("| variant | instructions in the loop | LDG | FFMA2 | FFMA | FSEL/SEL | LDS |")
    print("|---|---:|---:|---:|---:|---:|---:|")
    loops = {}
    for k in sorted(code):
        if "k_rows<" not in k:
            continue
        body = inner_loop(code[k])
        loops[k] = body
        ops = [re.sub(r"^@!?U?P\w+\s+", "", t).split()[0].split(".")[0] for _, t in body]
        cnt = lambda o: sum(1 for x in ops if x == o)
        print(f"| `{short(k)}` | {len(body)} | {cnt('LDG')} | {cnt('FFMA2')} | {cnt('FFMA')} | {cnt('FSEL') + cnt('SEL')} | {cnt('LDS')} |")
    print("\n(The skipping and partials variants hold both sides of their branches in the loop: the count is static, not "
          "what one iteration executes.)\n")
    for tag, title in (("k_rows<0, true, true, 0, false, false, false>", "cfg4 default on axis views: EA + ERT, 64-bit offsets, x-fastest array, scalar loads"),
                       ("k_rows<0, true, true, 0, false, false, true>", "cfg4 default on oblique views: the same with 16-byte row loads")):
        for k, body in loops.items():
            if tag in k:
                print(f"### {title}\n\n```")
                for a, t in body:
                    print(f"{a:04x}  {t}")
                print("```\n")


if __name__ == "__main__":
    main()
