"""Operand-reuse statistics of the fp64 instructions of one kernel of libfsp.so.

    python -m paper_2405_02603_b200.sass_reuse k_conv_z_fILi1024ELb0   [path/to/libfsp.so]

Why: on B200 a DFMA / DADD issues every 2 clocks per scheduler only while at most two of its 64-bit sources are NEW
register reads; a source is free when the instruction before it carried `.reuse` on the same register in the same
operand slot (operand reuse cache).  A DFMA with three new register reads issues every 3 clocks (fsp_ubench_fp64,
DESIGN.md "Three roofs").  This script reads `cuobjdump -sass` of the kernel whose mangled name contains the argument
and counts, per fp64 opcode, how many register sources each instruction has and how many of them are new reads.
"""
from __future__ import annotations

import os
import re
import subprocess
import sys

_INSTR = re.compile(r"^\s+/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)\s+(.*?);")
_REG = re.compile(r"(R\d+)(\.reuse)?")


def kernel_sass(lib: str, name_part: str) -> list[str]:
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    lines, keep = [], False
    for line in out.splitlines():
        if "Function :" in line:
            keep = name_part in line
        elif keep:
            lines.append(line)
    return lines


def reuse_statistics(lines) -> dict:
    prev: dict[int, str] = {}
    stat: dict[tuple, int] = {}
    for line in lines:
        m = _INSTR.match(line)
        if not m:
            continue
        op, args = m.group(1).split(".")[0], [a.strip() for a in m.group(2).split(",")]
        cur, regs, new = {}, 0, 0
        for slot, a in enumerate(args[1:]):
            r = _REG.search(a.replace("-", "").replace("|", ""))
            if not r or not a.lstrip("-|").startswith("R"):
                continue
            regs += 1
            if prev.get(slot) != r.group(1):
                new += 1
            if r.group(2):
                cur[slot] = r.group(1)
        if op in ("DFMA", "DADD", "DMUL"):
            stat[(op, regs, new)] = stat.get((op, regs, new), 0) + 1
        prev = cur
    return stat


def main(argv) -> int:
    if len(argv) < 2:
        print(__doc__)
        return 2
    lib = argv[2] if len(argv) > 2 else os.path.join(os.path.dirname(os.path.abspath(__file__)), "libfsp.so")
    lines = kernel_sass(lib, argv[1])
    if not lines:
        print("no kernel whose name contains", argv[1])
        return 1
    stat = reuse_statistics(lines)
    total = 0
    for (op, regs, new), c in sorted(stat.items()):
        print(f"{op}  register sources {regs}  new register reads {new}  count {c}")
        total += c
    three = {new: c for (op, regs, new), c in stat.items() if op == "DFMA" and regs == 3}
    n3 = sum(three.values())
    print("fp64 instructions (static):", total)
    if n3:
        print("DFMA with three register sources:", n3, " by new reads:",
              ", ".join(f"{k}: {v} ({v / n3:.3f})" for k, v in sorted(three.items())))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
