#!/usr/bin/env python
"""Count the FP64 instruction mix of the pair kernels' inner loops in the SASS of libbltc.so.

  python -m paper_2003_01833_b200.sass_count [--md]

For every near_kernel<R,OT,SUB,GUARD,KIND> / far_kernel<R,OT,SUB,GUARD,KIND,N1> instantiation the innermost loops that
contain MUFU.RSQ64H (one per (target, source-or-proxy) pair) are located through their backward branches
and their opcodes are counted (near: one loop per ZS variant, ZS = the r == 0 test is compiled in).  "pair" = one target against one source / proxy point, ALL OT orbitals of the tile;
flops = 2 DFMA + DMUL + DADD.  bench.py's FLOPS_PER_PAIR table holds the SUB = 1 rows.
Needs cuobjdump (CUDA toolkit); no GPU.
"""
from __future__ import annotations

import re
import subprocess
import sys

from . import build as _build


def kernels(lib):
    txt = subprocess.run(["cuobjdump", "-sass", lib], check=True, stdout=subprocess.PIPE, text=True).stdout
    cur, out = None, {}
    for line in txt.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            out[cur] = []
            continue
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m and cur:
            out[cur].append((int(m.group(1), 16), m.group(2).strip()))
    return out


def pair_loops(ins):
    """Innermost backward-branch loops that contain MUFU.RSQ64H (one per (target, source) pair)."""
    mufu = [a for a, t in ins if "MUFU.RSQ64H" in t]
    loops = []
    for a, t in ins:
        m = re.search(r"BRA(?:\.U)?\s+(?:!?U?P\d+,\s*)?0x([0-9a-f]+)", t)
        if not m:
            continue
        tgt = int(m.group(1), 16)
        if tgt < a and any(tgt <= x <= a for x in mufu):
            loops.append((tgt, a))
    inner = [l for l in loops if not any(o != l and l[0] <= o[0] and o[1] <= l[1] for o in loops)]
    return inner


def count(lib=None):
    lib = lib or _build.build()
    rows = []
    for name, ins in kernels(lib).items():
        m = re.search(r"(near_kernel|far_kernel)ILi(\d)ELi(\d)ELb([01])ELb([01])ELi(\d)E(?:Li(\d+)E)?", name)
        if not m:
            continue
        for lp in pair_loops(ins):
            body = [t for a, t in ins if lp[0] <= a <= lp[1]]
            ops = [re.sub(r"^@!?U?P\d+\s+", "", t).split()[0].split(".")[0] for t in body]
            pairs = sum("MUFU.RSQ64H" in t for t in body)
            zs = int(any("ISETP" in t and "0x7ff00000" in t for t in body))
            c = {k: ops.count(k) / pairs for k in ("DFMA", "DMUL", "DADD")}
            fp64 = c["DFMA"] + c["DMUL"] + c["DADD"]
            fma_pipe = sum(o in ("IMAD", "FFMA", "FMUL", "FADD") for o in ops) / pairs
            rows.append(dict(kernel=m.group(1), R=int(m.group(2)), OT=int(m.group(3)), SUB=int(m.group(4)),
                             GUARD=int(m.group(5)), KIND=int(m.group(6)), N1=int(m.group(7) or 0), ZS=zs, pairs=pairs, **c, fp64=fp64,
                             other=len(ops) / pairs - fp64, fma_pipe=fma_pipe,
                             flops=2 * c["DFMA"] + c["DMUL"] + c["DADD"]))
    rows.sort(key=lambda r: (r["KIND"], r["kernel"], r["R"], r["OT"], r["SUB"], r["GUARD"], r["N1"], r["ZS"]))
    return rows


def main():
    rows = count()
    hdr = ["kernel", "KIND", "R", "OT", "SUB", "GUARD", "N1", "ZS", "pairs", "DFMA", "DMUL", "DADD", "fp64", "other", "fma_pipe", "flops"]
    names = ["kernel", "KIND (0 Yukawa, 1 Coulomb)", "R", "OT", "SUB", "GUARD", "N1", "ZS", "pairs/iter", "DFMA/pair", "DMUL/pair", "DADD/pair", "FP64 instr/pair",
             "other instr/pair", "of which FMA-pipe", "flops/pair"]
    if "--md" in sys.argv:
        print("| " + " | ".join(names) + " |")
        print("|" + "---|" * len(names))
    for r in rows:
        cells = [f"{r[h]:.2f}" if isinstance(r[h], float) else str(r[h]) for h in hdr]
        print("| " + " | ".join(cells) + " |" if "--md" in sys.argv else "  ".join(cells))


if __name__ == "__main__":
    main()
