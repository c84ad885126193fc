"""Print the hot loops of the built library as SASS, with instruction counts per pipe class.

    python -m paper_2606_21784_b200.sass_report > profiles/r3_sass_hot_loops.md

The roofline argument of DESIGN.md 7.2 rests on how many 32x32->64 multiplies (IMAD.WIDE.U32 /
IMAD.HI.U32, the fmaheavy pipe) and how many instructions in all the generation loops execute per
agent event; tests/test_library_host.py checks those counts at test time, this module writes the
loops themselves down so that they can be read without rebuilding.  It only runs `cuobjdump -sass`
on libkineticsim.so and sorts text: nothing of the method's arithmetic is here.
"""
from __future__ import annotations

import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libkineticsim.so")

# (mangled-name fragment, title, ATOMS per loop iteration that marks a generation loop, which of those loops to
#  list in full: None = the shortest, else its index in address order)
KERNELS = [
    ("ks_decoupled_kernelILb0ELi1ELi4ELi160ELi7ELi2ELb0EEE",
     "ks_decoupled_kernel<0,1,4,160,7,2> -- the C4 / C2 headline plan: zero-intelligence, two steps per pass", 4, None),
    ("ks_persistent_kernelILi0ELi0ELb1EEE", "ks_persistent_kernel<0,0,1> -- PACKED4 zero-intelligence (one Philox block per 4 agents)", 8, None),
    ("ks_persistent_kernelILi2ELi0ELb0EEE", "ks_persistent_kernel<2,0,0> -- model 4, the paper's own agent rules (loops 0/3 noise, 1/4 momentum, 2/5 maker; "
     "0-2 the no-clamp forms)", 4, 0),
]


def classify(op: str) -> str:
    """Pipe class of one SASS opcode, as DESIGN.md 7.2 counts them."""
    if op.startswith("IMAD.WIDE") or op.startswith("IMAD.HI"):
        return "multiply (fmaheavy: IMAD.WIDE / IMAD.HI)"
    if op.startswith("IMAD"):
        return "other IMAD (fmaheavy/fmalite: MOV, SHL, IADD, 32-bit MAD forms)"
    if op.startswith("ATOMS") or op.startswith("RED") or op.startswith("ATOM"):
        return "shared-memory atomic (ATOMS)"
    if op.startswith(("LDS", "STS", "LDG", "STG", "LD.", "ST.", "LDC", "LDL", "STL", "ULDC")):
        return "load / store (LSU, constant)"
    if op.startswith(("LOP3", "SHF", "IADD3", "IADD", "LEA", "ISETP", "SEL", "IMNMX", "VIMNMX", "PRMT", "MOV", "SGXT", "PLOP3", "VIADD", "IABS", "FLO", "POPC", "BREV")):
        return "integer ALU (alu pipe: LOP3, SHF, IADD3, LEA, ISETP, SEL, MNMX, ...)"
    if op.startswith(("BRA", "BSSY", "BSYNC", "EXIT", "WARPSYNC", "BAR", "NOP", "CALL", "RET", "YIELD", "DEPBAR", "BREAK")):
        return "control (BRA, BAR, ...)"
    if op.startswith(("U", "R2UR", "S2UR", "VOTEU", "REDUX", "S2R", "CS2R", "SHFL", "VOTE", "MATCH")):
        return "uniform datapath / warp-wide (UIADD3, R2UR, SHFL, REDUX, ...)"
    return "other"


def loops_of(sass: str, fragment: str):
    bodies = [p for p in sass.split("Function : ") if fragment in p.split("\n", 1)[0]]
    if len(bodies) != 1:
        raise SystemExit("%d kernels match %r" % (len(bodies), fragment))
    ins = []
    for line in bodies[0].splitlines():
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2).strip()))
    loops = []
    for addr, text in ins:
        m = re.search(r"\bBRA\b.*?0x([0-9a-f]+)", text)
        if m and int(m.group(1), 16) <= addr:
            loops.append((int(m.group(1), 16), addr))
    inner = [(lo, hi) for lo, hi in loops if not any((l2, h2) != (lo, hi) and lo <= l2 and h2 <= hi for l2, h2 in loops)]
    return [[(a, t) for a, t in ins if lo <= a <= hi] for lo, hi in inner]


def opcode(text: str) -> str:
    t = re.sub(r"^@!?U?P\d+\s+", "", text)
    return t.split()[0]


def main() -> None:
    if not os.path.exists(LIB):
        raise SystemExit("build the library first: python -m paper_2606_21784_b200.build")
    sass = subprocess.check_output(["cuobjdump", "-sass", LIB]).decode()
    out = sys.stdout
    out.write("# r3 -- SASS of the generation hot loops (sm_100a), with instruction counts per pipe class\n\n")
    out.write("Command (no GPU needed; runs committed files only, after `python -m paper_2606_21784_b200.build`):\n\n")
    out.write("```\npython -m paper_2606_21784_b200.sass_report > profiles/r3_sass_hot_loops.md\n```\n\n")
    out.write("It runs `cuobjdump -sass paper_2606_21784_b200/libkineticsim.so`, takes the innermost loops (address range of a\n"
              "backward `BRA` that contains no other) of three kernels and keeps those that hold shared-memory atomics, i.e.\n"
              "the order-generation loops.  `tests/test_library_host.py` asserts the multiply counts on every build;\n"
              "`bench.py` turns events/s into executed multiplies/s with them (`roofline.executed_mults_per_event`).\n"
              "For each kernel ONE such loop is listed in full: the shortest (the no-clamp fast path the bulk of the events\n"
              "take), or for model 4 the no-clamp NOISE loop, which most of its agents run.\n\n")
    for fragment, title, min_atoms, which in KERNELS:
        loops = [l for l in loops_of(sass, fragment) if sum("ATOMS" in t for _, t in l) >= min_atoms]
        out.write("## `%s`\n\n" % title)
        out.write("| loop | instructions | ATOMS | IMAD.WIDE.U32 + IMAD.HI.U32 | multiplies per atomic | instructions per atomic |\n|---|---:|---:|---:|---:|---:|\n")
        for i, l in enumerate(loops):
            n = len(l)
            at = sum("ATOMS" in t for _, t in l)
            mu = sum(("IMAD.WIDE.U32" in t or "IMAD.HI.U32" in t) for _, t in l)
            out.write("| %d (0x%04x-0x%04x) | %d | %d | %d | %.2f | %.2f |\n" % (i, l[0][0], l[-1][0], n, at, mu, mu / at, n / at))
        out.write("\n")
        if not loops:
            continue
        pick = min(loops, key=len) if which is None else loops[which]
        counts = {}
        for _, t in pick:
            c = classify(opcode(t))
            counts[c] = counts.get(c, 0) + 1
        at = sum("ATOMS" in t for _, t in pick)
        out.write("%s loop (0x%04x-0x%04x), %d instructions for %d atomics, by pipe class:\n\n"
                  % ("Shortest" if which is None else "Loop %d," % which, pick[0][0], pick[-1][0], len(pick), at))
        out.write("| class | instructions | per atomic |\n|---|---:|---:|\n")
        for c, k in sorted(counts.items(), key=lambda kv: -kv[1]):
            out.write("| %s | %d | %.2f |\n" % (c, k, k / at))
        out.write("\n```\n")
        for a, t in pick:
            out.write("/*%04x*/  %s ;\n" % (a, t))
        out.write("```\n\n")


if __name__ == "__main__":
    main()
