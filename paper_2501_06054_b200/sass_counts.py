"""Executed instructions per class in a range of SASS lines of an Nsight Compute report (the counts behind
paper_2501_06054_b200/roofline.py; profiles/r2_instruction_counts.md states the ranges used).

    python -m paper_2501_06054_b200.sass_counts report.ncu-rep|source.csv[.gz] [--launch I] name:first:last:denominator ...
    python -m paper_2501_06054_b200.sass_counts report.ncu-rep --blocks        # runs of equal execution count

Classes: wide (IMAD.WIDE, IMAD.HI: 32x32->64 multiplies), imad (other integer multiplies), logic (LOP3, integer and
float compares, votes, selects, min/max), addr (integer adds, shifts, LEA, permutes, IMAD used as add/shift), fp64,
fp32, fp32x2 (packed FFMA2 / FMUL2 / FADD2: one instruction, two FP32 operations per lane), xu (MUFU, POPC, conversions), lsu (loads, stores, atomics), move (moves, uniform-datapath and constant loads),
ctl (branches, barriers, convergence, sleeps).  roofline.py counts wide, imad, logic, fp64, fp32, fp32x2 and xu as
algorithmic; addr, lsu, move and ctl are not.  `denominator` = executions of the unit the counts are per (e.g. the
execution count of the stage's first line times rows per step)."""
from __future__ import annotations

import collections
import csv
import subprocess
import sys

ORDER = ("wide", "imad", "logic", "addr", "fp64", "fp32", "fp32x2", "xu", "lsu", "move", "ctl")


def classify(full: str) -> str:
    p = full.split(".")
    op = p[0]
    if op == "IMAD":
        if "WIDE" in p or "HI" in p:
            return "wide"
        if "MOV" in p:
            return "move"
        if "IADD" in p or "SHL" in p or "U32" in p or "X" in p:
            return "addr"
        return "imad"
    if op in ("DFMA", "DMUL", "DADD", "DSETP"):
        return "fp64"
    if op in ("FFMA2", "FMUL2", "FADD2"):
        return "fp32x2"          # packed: one issue slot, two FP32 operations per lane (roofline.py: fma resource)
    if op in ("FFMA", "FMUL", "FADD", "HFMA2"):
        return "fp32"
    if op in ("MUFU", "POPC", "I2F", "F2I", "I2FP", "F2F", "FRND"):
        return "xu"
    if op in ("LOP3", "ISETP", "FSETP", "PLOP3", "VOTE", "SEL", "FSEL", "FMNMX", "VIMNMX"):
        return "logic"
    if op in ("IADD3", "VIADD", "LEA", "SHF", "PRMT"):
        return "addr"
    if op in ("LDS", "STS", "LDG", "STG", "RED", "REDG", "ATOM", "ATOMS", "ATOMG", "LDL", "STL"):
        return "lsu"
    if op in ("MOV", "UMOV", "CS2R", "S2R", "S2UR", "ULEA", "UIADD3", "ULOP3", "USEL", "UISETP", "UIMAD", "UFLO", "UPOPC",
              "VOTEU", "R2UR", "LDCU", "LDC", "REDUX", "USHF", "UPRMT"):
        return "move"
    return "ctl"


def load(rep: str, launch: int | None):
    if rep.endswith(".csv") or rep.endswith(".csv.gz"):   # an exported source page (ncu ... --page source --csv)
        import gzip
        text = (gzip.open(rep, "rt") if rep.endswith(".gz") else open(rep)).read()
        if launch:                                        # a multi-launch export: the launch-th "Kernel Name" section
            parts = text.split('"Kernel Name"')
            text = '"Kernel Name"' + parts[launch + 1]
    else:
        cmd = ["ncu", "-i", rep, "--page", "source", "--csv", "--print-source", "sass"]
        if launch is not None:
            cmd += ["--launch-skip", str(launch), "--launch-count", "1"]
        text = subprocess.run(cmd, capture_output=True, text=True).stdout
    rows = list(csv.reader(text.splitlines()))
    name = rows[0][1] if rows and len(rows[0]) > 1 else "?"
    hdr, data = rows[1], rows[2:]
    isrc, iex = hdr.index("Source"), hdr.index("Instructions Executed")
    out = []
    for r in data:
        if len(r) <= max(isrc, iex) or r[0] == "Kernel Name" or r[0] == "Address":
            break                                  # the next kernel of a multi-launch report
        out.append((r[isrc], int(r[iex] or 0)))
    return name, out


def main(argv):
    rep = argv[1]
    args = argv[2:]
    launch = None
    if "--launch" in args:
        i = args.index("--launch")
        launch = int(args[i + 1])
        del args[i:i + 2]
    name, d = load(rep, launch)
    print(f"kernel: {name}; {len(d)} SASS lines; {sum(e for _, e in d)} warp instructions executed")
    if "--blocks" in args:
        i = 0
        tot = sum(e for _, e in d)
        while i < len(d):
            j, e0 = i, d[i][1]
            while j < len(d) and abs(d[j][1] - e0) <= 0.02 * max(e0, 1):
                j += 1
            ex = sum(e for _, e in d[i:j])
            if ex > 0.003 * tot:
                print(f"lines {i:5d}-{j:5d}: {j - i:4d} lines x {e0:>11d} executions = {100 * ex / tot:5.1f} % of the instructions")
            i = j
        return
    for spec in args:
        label, a, b, den = spec.split(":")
        c = collections.Counter()
        for src, e in d[int(a):int(b)]:
            if e:
                t = src.split()
                c[classify(t[1] if t[0].startswith("@") else t[0])] += e / float(den)
        print(f"{label:14s} total {sum(c.values()):7.1f} | " + " ".join(f"{k}={c[k]:.1f}" for k in ORDER))


if __name__ == "__main__":
    main(sys.argv)
