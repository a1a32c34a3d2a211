"""Opcode counts per kernel of the built product library (evidence for profiles/, runs anywhere cuobjdump is installed).

    python -m paper_2606_04725_b200.sass_summary > profiles/<name>.md

Disassembles libnmpc_b200.so with `cuobjdump -sass` and counts, per kernel, the instructions that say what the kernel is
made of: DMMA (mma.sync.m8n8k4.f64: the fp64 tensor path -- tcgen05 has no f64 kind), DFMA / DMUL / DADD (fp64 vector
pipe), LDGSTS (cp.async), LDG / STG / LDS / STS, BAR, MUFU, ATOM / RED, and the Blackwell-only families UTMA* / UBLKCP (TMA)
and UTC*MMA (tcgen05), which this fp64 path does not use.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libnmpc_b200.so")
OPS = ("DMMA", "DFMA", "DMUL", "DADD", "MUFU", "LDGSTS", "LDG", "STG", "LDS", "STS", "BAR", "ATOM", "RED", "SHFL", "UTMA", "UBLKCP", "UTC")


def main():
    sass = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    arch = sorted(set(re.findall(r"arch = (sm_\w+)", sass)))
    counts, order, cur = collections.defaultdict(collections.Counter), [], None
    for ln in sass.splitlines():
        m = re.match(r"\s*Function : (\S+)", ln)
        if m:
            cur = m.group(1)
            order.append(cur)
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", ln)
        if m and cur:
            op = m.group(1)
            counts[cur]["total"] += 1
            for k in OPS:
                if op.startswith(k):
                    counts[cur][k] += 1
                    break
    demangled = subprocess.run(["cu++filt"] + order, capture_output=True, text=True).stdout.splitlines() if order else []
    names = {o: (d.split("(")[0].split("::")[-1] if d else o) for o, d in zip(order, demangled + [""] * len(order))}
    print(f"# SASS opcode counts per kernel, libnmpc_b200.so ({', '.join(arch)})")
    print()
    print("Command: `python -m paper_2606_04725_b200.sass_summary` (cuobjdump -sass on the built library; static instruction counts, "
          "not executed counts).")
    print()
    print("| kernel | instructions | " + " | ".join(OPS) + " |")
    print("|---|---|" + "---|" * len(OPS))
    for o in order:
        c = counts[o]
        print(f"| {names[o]} | {c['total']} | " + " | ".join(str(c[k]) for k in OPS) + " |")
    tot = collections.Counter()
    for o in order:
        tot.update(counts[o])
    print(f"| **all** | {tot['total']} | " + " | ".join(str(tot[k]) for k in OPS) + " |")
    print()
    print("DMMA is the tensor instruction of this path: `tcgen05.mma` has no f64 kind and `wgmma` does not exist on sm_100a. "
          "UTMA* / UBLKCP / UTC*MMA = 0: operands are staged with cp.async (LDGSTS), no TMA, no tcgen05.")


if __name__ == "__main__":
    main()
