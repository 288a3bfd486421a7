"""Opcode histogram of one kernel of libidg_b200.so (cuobjdump -sass), whole function and hottest loop.

    python -m paper_1609_03782_b200.sass_histogram 'idg_tma_kernelILi4ELi4ELi8ELi4ELi1ELb0ELb0E' [--loop N]

The "loop" is found structurally: the N-th largest span between a backward branch and its target (default: the
largest, which for the streaming kernels is the plane loop -- three unrolled ring phases).  Used to write the
listings under profiles/ (sass_*.txt); needs no GPU.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

LIB = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libidg_b200.so")


def function_sass(pattern: str) -> tuple:
    out = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    name, lines, take = None, [], False
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            if take:
                break
            take = pattern in m.group(1)
            name = m.group(1) if take else name
            continue
        if take:
            m = re.match(r"\s*/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
            if m:
                lines.append((int(m.group(1), 16), m.group(2).strip()))
    if not lines:
        raise SystemExit(f"no function matching {pattern!r} in {LIB}")
    return name, lines


def opcode(ins: str) -> str:
    t = ins.split()
    if t[0].startswith("@"):
        t = t[1:]
    return t[0]


def histogram(lines) -> collections.Counter:
    h = collections.Counter()
    for _, ins in lines:
        h[opcode(ins)] += 1
    return h


def loops(lines) -> list:
    """(start, end) address spans of backward branches, largest first."""
    spans = []
    for addr, ins in lines:
        m = re.search(r"\bBRA(?:\.[A-Z.]+)?\s+(?:[A-Z0-9!]+,\s*)?`?\(?(?:0x)?([0-9a-f]+)\)?", ins)
        if opcode(ins).startswith("BRA") and m:
            tgt = int(m.group(1), 16)
            if tgt < addr:
                spans.append((tgt, addr))
    return sorted(set(spans), key=lambda s: s[0] - s[1])


def report(pattern: str, which: int = 0) -> str:
    name, lines = function_sass(pattern)
    out = [f"kernel   {name}", f"library  {os.path.basename(LIB)}   ({len(lines)} SASS instructions)"]
    sp = loops(lines)
    groups = [("whole function", lines)]
    if sp:
        a, b = sp[min(which, len(sp) - 1)]
        groups.append((f"loop 0x{a:x}..0x{b:x} (backward branch span #{which})", [l for l in lines if a <= l[0] <= b]))
    for title, ls in groups:
        h = histogram(ls)
        out.append(f"\n== {title}: {len(ls)} instructions")
        cls = collections.Counter()
        for op, c in h.items():
            base = op.split(".")[0]
            kind = ("fp32 packed" if base in ("FFMA2", "FADD2", "FMUL2") else
                    "fp32 scalar" if base in ("FFMA", "FADD", "FMUL", "FSEL", "FMNMX", "FSETP") else
                    "mufu" if base == "MUFU" else
                    "shared ld/st" if base in ("LDS", "STS", "LDSM") else
                    "global ld/st" if base in ("LDG", "STG", "LD", "ST", "RED", "ATOMG") else
                    "tma/mbarrier" if base in ("UTMALDG", "SYNCS", "UTMASTG", "UBLKCP", "ELECT") else
                    "shuffle" if base == "SHFL" else
                    "barrier" if base in ("BAR", "WARPSYNC", "BSYNC", "BSSY") else
                    "branch" if base in ("BRA", "EXIT", "RET", "CALL", "JMP", "BRX") else
                    "move/select" if base in ("MOV", "SEL", "PRMT", "IMAD" if op.startswith("IMAD.MOV") else "_", "R2UR", "S2R", "S2UR", "CS2R", "UMOV") else
                    "integer/address")
            cls[kind] += c
        out.append("   by class: " + ", ".join(f"{k} {v}" for k, v in cls.most_common()))
        for op, c in h.most_common():
            out.append(f"   {c:6d}  {op}")
    return "\n".join(out)


if __name__ == "__main__":
    which = int(sys.argv[sys.argv.index("--loop") + 1]) if "--loop" in sys.argv else 0
    print(report(sys.argv[1], which))
