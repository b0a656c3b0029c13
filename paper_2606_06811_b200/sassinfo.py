"""Static instruction count of the Y-drop kernel's steady-state loop, read from the SASS of the
built library with cuobjdump ("instructions per cell counted from SASS").

The hot loop is one basic block holding 16 unrolled wavefront steps (16 message stores and 16 VIMNMX3, one per
cell and lane).  Two such blocks exist per kernel: the common one and the variant used while a strip
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
DPX = {"VIADDMNMX", "VIMNMX3"}       # Blackwell DPX; issue to the ALU pipe at the plain ALU rate (sfe_probe_int_issue)
FMA = {"IMAD"}
LSU = {"LDS", "STS", "LDG", "STG", "LDC", "LDCU", "ATOMG", "ATOMS", "RED"}

STEPS = 16.0      # wavefront steps per unrolled group (run_group16)

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
    """Returns dict(per_cell=I, alu=, fma=, lsu=, other=, hist=Counter) for the 16-step block."""
    name = "ydrop_kernelILb1ELb0EE" if traceback else "ydrop_kernelILb0ELb0EE"      # <TB, COOP = false>: the plain instantiation
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
    # the unrolled group may be split over a few adjacent basic blocks (ptxas peels its first step):
    # take every run of consecutive blocks that holds exactly STEPS message stores and STEPS VIMNMX3
    cnt = lambda b, name: sum(1 for _, op, _ in b if op == name)
    cand = []
    for i in range(len(blocks)):
        run, st, v3 = [], 0, 0
        for b in blocks[i:i + 4]:
            if run and b[0][0] != run[-1][0] + 16:
                break
            run += b; st += cnt(b, "STS"); v3 += cnt(b, "VIMNMX3")
            if st >= STEPS or v3 >= STEPS:
                break
        if st == STEPS and v3 >= STEPS and cnt(blocks[i], "VIMNMX3") > 0:
            cand.append(run)
    if not cand:
        raise RuntimeError(f"hot loop ({STEPS} message stores + VIMNMX3 per group) not found")
    blk = min(cand, key=len)
    hist = Counter(op for _, op, _ in blk)
    alu = sum(v for k, v in hist.items() if k in ALU)
    fma = sum(v for k, v in hist.items() if k in FMA)
    dpx = sum(v for k, v in hist.items() if k in DPX)
    lsu = sum(v for k, v in hist.items() if k in LSU)
    n = len(blk)
    return dict(per_cell=n / STEPS, alu=alu / STEPS, dpx=dpx / STEPS, fma=fma / STEPS, lsu=lsu / STEPS, other=(n - alu - fma - lsu) / STEPS,
                hist=dict(hist), n_blocks=len(cand))


if __name__ == "__main__":
    for tb in (True, False):
        h = hot_loop(tb)
        print("traceback" if tb else "score-only", {k: v for k, v in h.items() if k != "hist"})
        print("   ", h["hist"])
