"""Instruction-level summary of libbsl6d.so: per kernel family the SASS opcode histogram and the resource usage
(registers, spills, shared memory) of its instances.

    python -m paper_2303_05994_b200.sass_summary [--md] > profiles/<round>_sass_summary.md

Uses cuobjdump from the CUDA toolkit (no GPU needed).  What to look for (B200_PROFILING.md "What proves a
Blackwell-native kernel"): UTMALDG / UTMASTG = TMA bulk-tensor copies, SYNCS = mbarrier operations, UCGABAR = cluster
barriers, LDS/STS vs LDG/STG balance, DFMA counts; no HMMA / UTC*MMA anywhere (the op is a bandwidth-bound stencil).
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libbsl6d.so")
CUOBJDUMP = os.environ.get("CUOBJDUMP", "/usr/local/cuda/bin/cuobjdump")
SHOW = ("DFMA", "DMUL", "DADD", "LDG", "STG", "LDS", "STS", "LD", "ST", "LDL", "STL", "LDGSTS", "UTMALDG", "UTMASTG",
        "UBLKCP", "SYNCS", "UCGABAR", "BAR", "SHFL", "MAPA", "HMMA", "IMAD", "IADD3", "LOP3")


def family(name: str) -> str:
    m = re.search(r"bsl6d\d+(\w+?_kernel)", name)
    if m:
        return m.group(1)
    m = re.search(r"(\w+_kernel)", name)
    return m.group(1) if m else name[:40]


def demangle_args(name: str) -> str:
    m = re.search(r"_kernelI(.*?)E+v", name)
    if not m:
        return ""
    toks = re.findall(r"L[ib](\d+)E", m.group(1))
    return "<" + ",".join(toks) + ">"


def main():
    md = "--md" in sys.argv
    sass = subprocess.run([CUOBJDUMP, "-sass", LIB], capture_output=True, text=True, check=True).stdout
    res = subprocess.run([CUOBJDUMP, "--dump-resource-usage", LIB], capture_output=True, text=True, check=True).stdout
    ops = collections.defaultdict(collections.Counter)
    ninst = collections.Counter()
    fn = None
    for ln in sass.splitlines():
        s = ln.strip()
        if s.startswith("Function :"):
            fn = family(s.split(":", 1)[1].strip())
            ninst[fn] += 1
            continue
        m = re.match(r"/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", s)
        if m and fn:
            ops[fn][m.group(1).split(".")[0]] += 1
    usage = collections.defaultdict(list)
    cur = None
    for ln in res.splitlines():
        s = ln.strip()
        if s.startswith("Function "):
            cur = s.split()[1].rstrip(":")
        m = re.search(r"REG:(\d+) STACK:(\d+) SHARED:(\d+)", s)
        if m and cur:
            usage[family(cur)].append((demangle_args(cur), int(m.group(1)), int(m.group(2)), int(m.group(3))))
    print("# SASS summary of libbsl6d.so (sm_100a)\n")
    print("Command: `python -m paper_2303_05994_b200.sass_summary --md` (cuobjdump -sass / --dump-resource-usage on the "
          "in-tree library; no GPU needed).\n")
    print("## Opcode histogram per kernel family (all instances together)\n")
    cols = [c for c in SHOW if any(ops[f][c] for f in ops)]
    print("| family | instances | " + " | ".join(cols) + " |")
    print("|---|---|" + "---|" * len(cols))
    for f in sorted(ops):
        print(f"| {f} | {ninst[f]} | " + " | ".join(str(ops[f][c]) for c in cols) + " |")
    print("\n## Registers / spill stack / static shared memory per instance (template arguments as compiled)\n")
    for f in sorted(usage):
        rows = sorted(set(usage[f]))
        regs = [r[1] for r in rows]
        spills = [r for r in rows if r[2] > 0]
        print(f"* **{f}**: {len(rows)} instances, registers {min(regs)}-{max(regs)}; "
              f"{'no instance spills' if not spills else 'spilling instances: ' + ', '.join(f'{a} ({st} B stack, {rg} regs)' for a, rg, st, _ in spills[:12])}")
    print()
    tc = [f for f in ops if any(k.startswith(("HMMA", "UTCHMMA", "UTCQMMA", "HGMMA", "IMMA", "DMMA")) for k in ops[f])]
    print("Tensor-core instructions: " + ("none (as intended: bandwidth-bound stencil, no dense contraction)" if not tc
                                          else ", ".join(tc)))


if __name__ == "__main__":
    main()
