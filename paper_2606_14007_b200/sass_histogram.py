"""SASS opcode histogram of libvx.so's kernels (cuobjdump -sass), per kernel.

    python -m paper_2606_14007_b200.sass_histogram [kernel-name-regex] [--per N]

The roofline of stage 1 is stated in instructions per hash; this prints what ptxas
actually emitted so that the numbers can be re-derived: opcode counts of the matching kernels, each
divided by N (`--per 4`: vx_k_hash_scatter hashes 4 nonces per thread in straight-line code).
The pipe column follows the issue rates measured by bench.py --probe-alu (profiles/r02_alu_probe.md):
LOP3 / SHF / PRMT issue at 16 lanes per clock per SM sub-partition (the half-rate integer pipe, "alu"),
IMAD at 16 (the FMA pipe, "fma"), IADD3 at 32 ("add": both).
"""
from __future__ import annotations

import argparse
import collections
import re
import subprocess
import sys

from . import build as _build

ALU = ("LOP3", "SHF", "PRMT", "ISETP", "SEL", "LEA", "IABS", "BREV", "FLO", "POPC", "VIADD", "VIMNMX", "IMNMX",
       "LOP", "SGXT", "BMSK", "PLOP3", "P2R", "R2P", "IADD", "MOV", "CS2R")
FMA = ("IMAD", "FFMA", "FMUL", "FADD")


def pipe_of(op: str) -> str:
    base = op.split(".")[0]
    if base == "IADD3":
        return "add"
    if base in FMA:
        return "fma"
    if base in ALU:
        return "alu"
    if base in ("LDG", "STG", "LDS", "STS", "ATOMS", "ATOMG", "ATOM", "RED", "LDC", "LDCU", "LD", "ST", "LDL", "STL"):
        return "lsu"
    return "other"


def histograms(pattern: str):
    text = subprocess.check_output(["cuobjdump", "-sass", _build.LIB], text=True)
    out = {}
    name = None
    for line in text.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            if re.search(pattern, name):
                out[name] = collections.Counter()
            else:
                name = None
            continue
        if name is None:
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if m:
            out[name][m.group(1)] += 1
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("pattern", nargs="?", default="vx_k_hash_scatterILb0|vx_k_sort_matchILi512ELi9ELi12ELi2ELb0")
    ap.add_argument("--per", type=float, default=1.0, help="divide the counts by this (work items per thread)")
    args = ap.parse_args(argv)
    for name, hist in histograms(args.pattern).items():
        demangled = subprocess.run(["c++filt", name], capture_output=True, text=True).stdout.strip() or name
        total = sum(hist.values())
        print(f"## {demangled}\n# {total} SASS instructions ({total / args.per:.1f} per work item, --per {args.per:g})")
        pipes = collections.Counter()
        for op, n in hist.items():
            pipes[pipe_of(op)] += n
        print("# by pipe: " + ", ".join(f"{p} {n} ({n / args.per:.1f})" for p, n in sorted(pipes.items(), key=lambda t: -t[1])))
        for op, n in sorted(hist.items(), key=lambda t: -t[1]):
            print(f"{n:7d} {n / args.per:9.2f}  {pipe_of(op):5s} {op}")
        print()
    return 0


if __name__ == "__main__":
    sys.exit(main())
