"""Opcode summary of the built library, kept under profiles/ as evidence of what the kernels are made of.

    python -m paper_1612_06592_b200.sass_summary [--lib PATH] > profiles/sass_summary.md

Runs `cuobjdump -sass` and `cuobjdump -res-usage` on liblofar_moon.so (no GPU needed) and prints, per kernel, the
static count of the opcodes that identify the hardware paths in use: UTCHMMA / LDTM / UTCBAR (tcgen05 MMA, TMEM
load, tcgen05 commit), UBLKCP / SYNCS (bulk asynchronous copy and its mbarrier), packed fp32x2 arithmetic
(FFMA2 / FADD2), scalar FFMA, shared-memory and shuffle traffic, registers and static shared memory.  Counts are of
instructions in the binary, not of executed instructions (those are in the ncu summaries)."""
from __future__ import annotations

import os
import re
import subprocess
import sys
from collections import Counter, OrderedDict

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liblofar_moon.so")
OPS = ["UTCHMMA", "LDTM", "UTCBAR", "UBLKCP", "SYNCS", "FFMA2", "FADD2", "FFMA", "FMUL", "FADD", "LDS", "STS", "SHFL",
       "LDG", "STG", "BAR", "DFMA", "DADD"]


def demangle(name: str) -> str:
    """beamform_kernel<24, 2, false> from the mangled symbol (c++filt), without namespaces and arguments."""
    try:
        full = subprocess.run(["c++filt", name], capture_output=True, text=True, check=True).stdout.strip()
    except (OSError, subprocess.CalledProcessError):
        return name
    full = re.sub(r"\(anonymous namespace\)::|lofar::", "", full)
    depth = 0
    for i, ch in enumerate(full):                      # cut the argument list: the first '(' outside template brackets
        depth += ch == "<"
        depth -= ch == ">"
        if ch == "(" and depth == 0:
            return full[:i].replace("void ", "")
    return full


def main(argv):
    lib = argv[argv.index("--lib") + 1] if "--lib" in argv else LIB
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    res = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    usage = {}
    cur = None
    for ln in res.splitlines():
        m = re.search(r"Function (\S+):", ln)
        if m:
            cur = demangle(m.group(1))
            continue
        m = re.search(r"REG:(\d+).*?SHARED:(\d+)", ln)
        if m and cur:
            usage[cur] = (int(m.group(1)), int(m.group(2)))
            cur = None
    kernels: "OrderedDict[str, Counter]" = OrderedDict()
    k = None
    for ln in sass.splitlines():
        m = re.search(r"Function : (\S+)", ln)
        if m:
            k = demangle(m.group(1))
            kernels[k] = Counter()
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", ln)
        if m and k:
            kernels[k][m.group(1)] += 1
            kernels[k]["_total"] += 1
    print("# SASS opcode summary of paper_1612_06592_b200/liblofar_moon.so (sm_100a)\n")
    print("Command (no GPU needed; regenerate whenever a kernel changes):\n")
    print("```\npython -m paper_1612_06592_b200.build && python -m paper_1612_06592_b200.sass_summary > profiles/sass_summary.md\n```\n")
    print("Static instruction counts from `cuobjdump -sass`, registers / static shared memory from `cuobjdump -res-usage` "
          "(dynamic shared memory is set at launch: 211 KB for ippf_kernel / rescan_kernel, 23 KB for beamform_tc_kernel "
          "at 24 beams).\n")
    print("| kernel | instr | regs | " + " | ".join(OPS) + " |")
    print("|---|---|---|" + "---|" * len(OPS))
    for name, c in kernels.items():
        regs = usage.get(name, ("?", "?"))[0]
        print(f"| {name} | {c['_total']} | {regs} | " + " | ".join(str(c.get(o, 0)) for o in OPS) + " |")
    print("\nReading: `beamform_tc_kernel` is the only kernel with tcgen05 (UTCHMMA = tcgen05.mma, LDTM = tcgen05.ld, "
          "UTCBAR = tcgen05.commit); `ippf_kernel` stages its input with the bulk-copy engine (UBLKCP = cp.async.bulk, "
          "SYNCS = mbarrier arrive/try_wait) and does its arithmetic in packed fp32x2 (FFMA2, FADD2); no kernel uses "
          "wgmma/mma.sync.")


if __name__ == "__main__":
    main(sys.argv[1:])
