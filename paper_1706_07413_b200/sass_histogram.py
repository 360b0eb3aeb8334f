"""Static opcode histogram of the Runge-Kutta stage loop of the resident kernel, from the in-tree build objects.

    python -m paper_1706_07413_b200.sass_histogram [CL ...]        # default: 2 1  (cfg2's build and the one-CTA build)

Reads `cuobjdump -sass` of paper_1706_07413_b200/build/adsc_resident3_*.o (made by paper_1706_07413_b200.build), takes
k_resident3<8, 256, true, CL, false, 4> (dynamical metric, classical RK4), finds its stage loop (the largest loop nested
inside the largest loop, which is the step loop) and counts the instructions of the loop body by class, per
thread-stage and per point-stage (a thread owns 8 points).  STATIC counts: all four tiers of the exponential are in
the body and one of them runs, so the executed FP64 share is lower than the static one (ncu: ~52 FP64 instructions
per point-stage executed on cfg2 against ~89 in the listing).  A diagnosis tool for profiles/; nothing imports it.
"""
from __future__ import annotations

import collections
import glob
import os
import re
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))

CLASSES = [
    ("FP64 arithmetic (DFMA/DMUL/DADD)", {"DFMA", "DMUL", "DADD"}),
    ("FP64 compare (DSETP/DMNMX)", {"DSETP", "DMNMX"}),
    ("FP32 / convert / MUFU", {"MUFU", "F2F", "I2F", "F2I", "FSEL", "FMUL", "FFMA", "FADD", "FSETP", "I2FP", "F2FP"}),
    ("SHFL", {"SHFL"}),
    ("SYNCS / STAS / fences (mbarrier, DSMEM)", {"SYNCS", "STAS", "MEMBAR", "FENCE", "UCGABAR_ARV", "UCGABAR_WAIT", "CCTL",
                                                 "ERRBAR", "ATOMS", "ATOM", "RED"}),
    ("BAR / WARPSYNC", {"BAR", "WARPSYNC", "NANOSLEEP", "YIELD"}),
    ("global / local memory", {"LDG", "STG", "LD", "ST", "LDL", "STL"}),
    ("constant loads (LDC/ULDC)", {"LDC", "ULDC", "LDCU"}),
    ("moves / select / predicate", {"MOV", "UMOV", "R2UR", "S2R", "S2UR", "CS2R", "PRMT", "SEL", "USEL", "R2P", "P2R", "PLOP3",
                                    "UPLOP3", "VOTE", "VOTEU", "MOVM"}),
    ("control (BRA/BSSY/BSYNC)", {"BRA", "BSSY", "BSYNC", "EXIT", "NOP", "BRX", "CALL", "RET", "BREAK", "BMOV", "BPT"}),
]


def classify(op: str) -> str:
    parts = op.split(".")
    if parts[0] in ("LDS", "STS"):
        return parts[0] + "." + (parts[1] if len(parts) > 1 and parts[1] in ("64", "128") else "32")
    for name, ops in CLASSES:
        if parts[0] in ops:
            return name
    return "integer ALU (IADD3/IMAD/LEA/LOP3/SHF/ISETP/...)"


def stage_loop(cl: int):
    """(instructions of the stage loop body as (address, opcode, text), function name)"""
    fn = f"_ZN4adsc11k_resident3ILi8ELi256ELb1ELi{cl}ELb0ELi4EEEvNS_9ResParamsE"
    for obj in sorted(glob.glob(os.path.join(_HERE, "build", "adsc_resident3_*.o"))):
        out = subprocess.run(["cuobjdump", "-sass", "-fun", fn, obj], capture_output=True, text=True).stdout
        ins = []
        for line in out.splitlines():
            m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
            if m:
                t = m.group(2).split()
                ins.append((int(m.group(1), 16), t[1] if t[0].startswith("@") else t[0], m.group(2)))
        if not ins:
            continue
        loops = []
        for a, op, txt in ins:
            m = re.search(r"0x([0-9a-f]+)", txt) if op.startswith("BRA") else None
            if m and int(m.group(1), 16) <= a:
                loops.append((int(m.group(1), 16), a))
        loops.sort(key=lambda l: l[0] - l[1])
        outer = loops[0]
        lo, hi = next(l for l in loops[1:] if outer[0] <= l[0] and l[1] <= outer[1])
        return [i for i in ins if lo <= i[0] <= hi], fn, (lo, hi), os.path.basename(obj)
    raise SystemExit(f"{fn} not found: build the library first (python -m paper_1706_07413_b200.build)")


def main(argv):
    cls = [int(a) for a in argv] or [2, 1]
    res, tot = {}, {}
    for cl in cls:
        body, fn, (lo, hi), obj = stage_loop(cl)
        res[cl] = collections.Counter(classify(op) for _, op, _ in body)
        tot[cl] = len(body)
        print(f"CL={cl}: {fn} in build/{obj}, stage loop 0x{lo:x}..0x{hi:x}, {len(body)} instructions")
    keys = sorted({k for c in res.values() for k in c}, key=lambda k: -res[cls[0]][k])
    print("\n| class | " + " | ".join(f"CL={c}: per thread-stage | per point-stage | share" for c in cls)
          + (f" | CL={cls[0]} minus CL={cls[1]} |" if len(cls) > 1 else " |"))
    print("|---|" + "---|---|---|" * len(cls) + ("---|" if len(cls) > 1 else ""))
    for k in keys:
        row = " | ".join(f"{res[c][k]} | {res[c][k] / 8:.1f} | {100 * res[c][k] / tot[c]:.1f} %" for c in cls)
        print(f"| {k} | {row}" + (f" | {res[cls[0]][k] - res[cls[1]][k]:+d} |" if len(cls) > 1 else " |"))
    row = " | ".join(f"{tot[c]} | {tot[c] / 8:.1f} | " for c in cls)
    print(f"| **total** | {row}" + (f" | {tot[cls[0]] - tot[cls[1]]:+d} |" if len(cls) > 1 else " |"))


if __name__ == "__main__":
    main(sys.argv[1:])
