"""Static instruction count of the Y-drop kernel's steady-state loop, read from the SASS of the
built library with cuobjdump ("instructions per cell counted from SASS").

The hot loop is one basic block holding 8 unrolled wavefront steps (8 VIMNMX3, one per cell and
lane).  Two such blocks exist per kernel: the common one and the variant used while a strip
crosses the right edge of the DP matrix; the common one is the shorter.
"""
from __future__ import annotations

import os
import re
import subprocess
from collections import Counter

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(_HERE, "libsfe.so")

ALU = {"ISETP", "SEL", "IADD3", "VIADD", "VIADDMNMX", "VIMNMX3", "VIMNMX", "PRMT", "LOP3", "SHF", "LEA", "MOV",
       "IABS", "FLO", "POPC", "BREV", "PLOP3", "P2R", "R2P", "IADD"}
FMA = {"IMAD"}
LSU = {"LDS", "STS", "LDG", "STG", "LDC", "LDCU", "ATOMG", "ATOMS", "RED"}

_INS = re.compile(r"^\s*/\*([0-9a-f]{4,6})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)((?:\.[A-Z0-9_]+)*)")


def _sass(kernel_substr: str) -> list[tuple[int, str, str]]:
    out = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    ins, on = [], False
    for ln in out.splitlines():
        if "Function :" in ln:
            on = kernel_substr in ln
            continue
        if not on:
            continue
        m = _INS.match(ln)
        if m:
            ins.append((int(m.group(1), 16), m.group(2), ln))
    return ins


def hot_loop(traceback: bool = True) -> dict:
    """Returns dict(per_cell=I, alu=, fma=, lsu=, other=, hist=Counter) for the 8-step block."""
    name = "ydrop_kernelILb1EE" if traceback else "ydrop_kernelILb0EE"
    ins = _sass(name)
    if not ins:
        raise RuntimeError(f"kernel {name} not found in {LIB}")
    # split into basic blocks at control-flow instructions and branch targets
    targets = set()
    for _, op, ln in ins:
        if op in ("BRA", "BSSY"):
            m = re.search(r"0x([0-9a-f]+)\s*;", ln)
            if m:
                targets.add(int(m.group(1), 16))
    blocks, cur = [], []
    for a, op, ln in ins:
        if a in targets and cur:
            blocks.append(cur); cur = []
        cur.append((a, op, ln))
        if op in ("BRA", "EXIT", "RET", "BSYNC"):
            blocks.append(cur); cur = []
    if cur:
        blocks.append(cur)
    cand = [b for b in blocks if sum(1 for _, op, _ in b if op == "VIMNMX3") == 8]
    if not cand:
        raise RuntimeError("hot loop (8 x VIMNMX3) not found")
    blk = min(cand, key=len)
    hist = Counter(op for _, op, _ in blk)
    alu = sum(v for k, v in hist.items() if k in ALU)
    fma = sum(v for k, v in hist.items() if k in FMA)
    lsu = sum(v for k, v in hist.items() if k in LSU)
    n = len(blk)
    return dict(per_cell=n / 8.0, alu=alu / 8.0, fma=fma / 8.0, lsu=lsu / 8.0, other=(n - alu - fma - lsu) / 8.0,
                hist=dict(hist), n_blocks=len(cand))


if __name__ == "__main__":
    for tb in (True, False):
        h = hot_loop(tb)
        print("traceback" if tb else "score-only", {k: v for k, v in h.items() if k != "hist"})
        print("   ", h["hist"])
