"""Per-kernel resource table and SASS opcode histogram of liblbmk.so, as markdown on stdout.

    python -m paper_2607_05668_b200.resource_table > profiles/r2_resource_usage.md

Registers, spill stores/loads, stack frame and shared memory come from ptxas (`-Xptxas -v`, the logs `_build.py` keeps in
`paper_2607_05668_b200/build/*.ptxas.log`; the library is rebuilt with --force first so that they belong to the current sources);
the opcode histograms come from `cuobjdump -sass` of the built library for the kernels the roofline numbers are quoted on.
No GPU needed.  What the paper reports for its own kernels (RTX A5000): 255 registers and 32 / 104 B of spills for the 18-field
MHD and the 14-field HCNSF kernels.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

from . import _build

HEADLINE = [  # (label, unit, regex on the demangled-ish mangled name)
    ("c4 NSF3D f32, pull, forcing on", "sys_nsf3d", r"collide_stream_nodeINS_8SysNsf3DIfEEfLi0ELb1ELi64ELi6ELb0ELb0E"),
    ("c4 NSF3D f32, pull, forcing off", "sys_nsf3d", r"collide_stream_nodeINS_8SysNsf3DIfEEfLi0ELb0ELi64ELi6ELb0ELb0E"),
    ("c5 MHD3D f32, pull", "sys_mhd3d", r"collide_stream_nodeINS_8SysMhd3DIfEEfLi0ELb0ELi64ELi4ELb0ELb0E"),
    ("c3 Euler2D f32, pull", "sys_euler2d", r"collide_stream_nodeINS_10SysEuler2DIfEEfLi0ELb0ELi128ELi1ELb0ELb0E"),
    ("HCNSF f32, pull", "sys_hcnsf3d", r"collide_stream_nodeINS_10SysHcnsf3DIfEEfLi0ELb0ELi64ELi6ELb0ELb0E"),
    ("HCNSF f64, pull", "sys_hcnsf3d", r"collide_stream_nodeINS_10SysHcnsf3DIdEEdLi0ELb0ELi128ELi1ELb0ELb0E"),
    ("MHD2D f32, pull, forcing off", "sys_mhd2d", r"collide_stream_nodeINS_8SysMhd2DIfEEfLi0ELb0ELi128ELi3ELb0ELb0E"),
    ("MHD2D f32, pull, forcing on", "sys_mhd2d", r"collide_stream_nodeINS_8SysMhd2DIfEEfLi0ELb1ELi128ELi3ELb0ELb0E"),
    ("MHD2D f64, pull, forcing off", "sys_mhd2d", r"collide_stream_nodeINS_8SysMhd2DIdEEdLi0ELb0ELi128ELi1ELb0ELb0E"),
    ("c2 SWE f64, pull, forcing on (per launch)", "sys_swe2d", r"collide_stream_nodeINS_8SysSwe2DIdEEdLi0ELb1ELi128ELi1ELb0ELb0E"),
    ("c2 SWE f64, persistent (fat blocks, the one c2 runs), forcing on", "sys_swe2d", r"collide_stream_persistent_fatINS_8SysSwe2DIdEEdLb1E"),
    ("c2 SWE f64, persistent (thin blocks), forcing on", "sys_swe2d", r"collide_stream_persistentINS_8SysSwe2DIdEEdLb1E"),
    ("c2 SWE f64, SM-resident (AA in shared memory), forcing on", "sys_swe2d", r"collide_stream_residentINS_8SysSwe2DIdEEdLb1ELi512E"),
    ("c1 advection f64, cluster-resident", "sys_advection2d", r"collide_stream_clusterINS_14SysAdvection2DIdEEdEE"),
    ("c1 advection f64, persistent", "sys_advection2d", r"collide_stream_persistentINS_14SysAdvection2DIdEEdLb0E"),
    ("c4 NSF3D f32, TRT, forcing on", "sys_nsf3d", r"collide_stream_nodeINS_8SysNsf3DIfEEfLi0ELb1ELi64ELi6ELb1ELb0E"),
]


def parse_ptxas(path):
    """{mangled name: dict(regs, spill_st, spill_ld, stack, smem)}"""
    out, name = {}, None
    rec = {}
    for ln in open(path):
        m = re.search(r"Function properties for (\S+)", ln)
        if m:
            name, rec = m.group(1), {}
            continue
        m = re.search(r"(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads", ln)
        if m and name:
            rec.update(stack=int(m.group(1)), spill_st=int(m.group(2)), spill_ld=int(m.group(3)))
            continue
        m = re.search(r"Used (\d+) registers", ln)
        if m and name:
            rec["regs"] = int(m.group(1))
            ms = re.search(r"(\d+) bytes smem", ln)
            rec["smem"] = int(ms.group(1)) if ms else 0
            out[name] = rec
            name = None
    return out


def sass_histogram(lib, mangled):
    r = subprocess.run(["cuobjdump", "-sass", "-fun", mangled, lib], capture_output=True, text=True)
    ops = collections.Counter()
    for ln in r.stdout.splitlines():
        m = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", ln)
        if m:
            ops[m.group(1).split(".")[0]] += 1
    return ops


def main():
    lib = _build.build(force=True)
    logs = {}
    for u in _build.UNITS:
        logs[u] = parse_ptxas(os.path.join(_build.OBJ, u + ".ptxas.log"))
    print("# Round 2 — registers, spills, shared memory and SASS opcode mix of the step kernels (sm_100a)\n")
    print("Command: `python -m paper_2607_05668_b200.resource_table > profiles/r2_resource_usage.md` (rebuilds the library with")
    print("`nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -Xptxas -v`, parses ptxas' output, runs `cuobjdump -sass`).\n")
    print("| kernel | registers | spill stores / loads (B) | stack (B) | static smem (B) | SASS instructions | top opcodes |")
    print("|---|---|---|---|---|---|---|")
    for label, unit, pat in HEADLINE:
        hits = [(n, r) for n, r in logs[unit].items() if re.search(pat, n)]
        if not hits:
            print(f"| {label} | (not found: {pat}) | | | | | |")
            continue
        n, r = hits[0]
        ops = sass_histogram(lib, n)
        top = ", ".join(f"{k} {v}" for k, v in ops.most_common(10))
        print(f"| {label} | {r['regs']} | {r['spill_st']} / {r['spill_ld']} | {r['stack']} | {r['smem']} | {sum(ops.values())} | {top} |")
    print("\n## Every collide_stream_* instantiation\n")
    print("| unit | kernel (mangled, shortened) | registers | spill st / ld (B) |")
    print("|---|---|---|---|")
    for u in _build.UNITS:
        for n, r in sorted(logs[u].items()):
            if "collide_stream" in n:
                short = re.sub(r"^_ZN4lbmk\d+", "", n)[:88]
                print(f"| {u} | `{short}` | {r['regs']} | {r['spill_st']} / {r['spill_ld']} |")


if __name__ == "__main__":
    sys.exit(main())
