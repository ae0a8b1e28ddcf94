"""Resource and SASS summary of libah_b200.so, for profiles/ (no GPU needed).

    python -m paper_2005_14454_b200.sass_summary > profiles/rNN_sass_summary.md

Per kernel: registers, stack, static shared memory (cuobjdump -res-usage) and the count of the SASS mnemonics that
carry the design: UBLKCP (bulk-TMA copies), SYNCS (mbarrier), ELECT, FFMA2/FMUL2/FADD2 (packed fp32), FFMA/FMUL/FADD,
MUFU, F2F/F2I (conversion pipe), D* (fp64), LDL/STL (spills), LDS/STS, LDG/STG, BAR.
"""
from __future__ import annotations

import re
import subprocess
import sys
from collections import Counter

from .build import LIB, build

MNEMONICS = ("UBLKCP", "SYNCS", "ELECT", "FFMA2", "FMUL2", "FADD2", "FFMA", "FMUL", "FADD", "MUFU", "F2F", "F2I",
             "DFMA", "DADD", "DMUL", "LDL", "STL", "LDS", "STS", "LDG", "STG", "BAR", "UTCHMMA", "UTCQMMA")


def demangle(names):
    out = subprocess.run(["c++filt"] + list(names), capture_output=True, text=True).stdout.splitlines()
    return dict(zip(names, out))


def main():
    build()
    res = subprocess.run(["cuobjdump", "-res-usage", str(LIB)], capture_output=True, text=True, check=True).stdout
    usage = {}
    cur = None
    for line in res.splitlines():
        m = re.search(r"Function (\S+):", line)
        if m:
            cur = m.group(1)
            continue
        if cur and "REG:" in line:
            usage[cur] = dict(re.findall(r"(\w+):(\d+)", line))
            cur = None
    sass = subprocess.run(["cuobjdump", "-sass", str(LIB)], capture_output=True, text=True, check=True).stdout
    counts, total = {}, Counter()
    cur = None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            counts[cur] = Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,6}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", line)
        if m and cur:
            counts[cur][m.group(1)] += 1
            total[cur] += 1
    names = demangle(sorted(counts))
    print("# SASS / resource summary of libah_b200.so (sm_100a)\n")
    print("Made by `python -m paper_2005_14454_b200.sass_summary` (cuobjdump -res-usage, cuobjdump -sass; no GPU).\n")
    print("| kernel | REG | STACK | SHARED (static) | SASS instr | " + " | ".join(MNEMONICS) + " |")
    print("|---|" + "---|" * (4 + len(MNEMONICS)))
    for mangled in sorted(counts, key=lambda k: names[k]):
        u = usage.get(mangled, {})
        short = re.sub(r"ah::\(anonymous namespace\)::|ah::", "", names[mangled])
        short = re.sub(r"\(.*", "", short).replace("void ", "")
        row = [short, u.get("REG", "?"), u.get("STACK", "?"), u.get("SHARED", "?"), str(total[mangled])]
        row += [str(counts[mangled].get(k, 0)) for k in MNEMONICS]
        print("| " + " | ".join(row) + " |")
    print("\nNo UTC*MMA (tcgen05) is expected anywhere: the path is a stencil, not a contraction (DESIGN.md).")
    return 0


if __name__ == "__main__":
    sys.exit(main())
