"""Opcode histogram of the step loop of a persistent kernel, from `cuobjdump -sass` of the built library.

    python tests/sass_histogram.py [bulk|coop]

The step loop is the innermost loop that contains the Runge-Kutta attempt: the backward branch with the smallest
span among those that enclose at least six MUFU.RCP64H (one reciprocal per stage).  Prints the FP64-pipe count
(DFMA + DMUL + DADD + DSETP), the other opcodes and the local-memory instructions (LDL / STL: spills, must be 0).
The count is static: rarely taken branches inside the loop are included.  Test infrastructure (tests/test_host_logic.py) and reporting
only: nothing here is used by the library.
"""
from __future__ import annotations

import collections
import re
import subprocess
import sys
from pathlib import Path

LIB = Path(__file__).resolve().parent.parent / "paper_2509_15117_b200" / "libia_b200.so"
KERNELS = {"bulk": "ia_persistent_kernelILi1ELi2", "coop": "ia_persistent_kernelILi3ELi1"}


def instructions(kernel: str):
    out = subprocess.run(["cuobjdump", "-sass", str(LIB)], capture_output=True, text=True, check=True).stdout
    ins, inside = [], False
    for line in out.splitlines():
        if "Function :" in line:
            inside = KERNELS[kernel] in line
            continue
        if not inside:
            continue
        m = re.match(r"\s+/\*([0-9a-f]{4,6})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), re.sub(r"^@!?U?P\d+\s+", "", m.group(2))))
    return ins


def step_loop(ins):
    best = None
    for addr, text in ins:
        m = re.search(r"\bBRA\b.*?(0x[0-9a-f]+)", text)
        if not m:
            continue
        tgt = int(m.group(1), 16)
        if tgt >= addr:
            continue
        body = [t for a, t in ins if tgt <= a <= addr]
        if sum(t.startswith("MUFU.RCP64H") for t in body) >= 6 and (best is None or len(body) < len(best[2])):
            best = (tgt, addr, body)
    return best


def main():
    kernel = sys.argv[1] if len(sys.argv) > 1 else "bulk"
    ins = instructions(kernel)
    lo, hi, body = step_loop(ins)
    hist = collections.Counter(t.split()[0].split(".")[0] for t in body)
    fp64 = sum(hist[k] for k in ("DFMA", "DMUL", "DADD", "DSETP"))
    whole = collections.Counter(t.split()[0].split(".")[0] for _, t in ins)
    print(f"kernel {KERNELS[kernel]}: {len(ins)} instructions; step loop {lo:#x}..{hi:#x}: {len(body)} instructions")
    print(f"  FP64 pipe: {fp64} = " + " + ".join(f"{hist[k]} {k}" for k in ("DFMA", "DMUL", "DADD", "DSETP")))
    print(f"  other: {len(body) - fp64} = " + ", ".join(f"{v} {k}" for k, v in hist.most_common()
                                                         if k not in ("DFMA", "DMUL", "DADD", "DSETP")))
    print(f"  local memory in the whole kernel: {whole['LDL']} LDL, {whole['STL']} STL")
    print(f"  flops per attempted step counted from SASS: {2 * hist['DFMA'] + hist['DMUL'] + hist['DADD']}")
    print(f"  STATIC count: the loop body holds both branches of the error norm (the general tree is not taken in these "
          f"units) and the rarely taken event / termination branch; the instructions a step executes are counted by "
          f"ncu (profiles/r02_summary.md section 3, profiles/r03_ncu.md)")
    print(f"  issue slots if every instruction of the body ran: 2 x {fp64} + {len(body) - fp64} = "
          f"{2 * fp64 + len(body) - fp64}")


if __name__ == "__main__":
    main()
