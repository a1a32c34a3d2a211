"""Markdown summaries of ncu exports (evidence for profiles/; reads text files only, runs anywhere).

    python -m paper_2606_04725_b200.ncu_summary launches gpurun_out/<launch list>.csv  > profiles/<name>.md
    python -m paper_2606_04725_b200.ncu_summary raw      profiles/<raw page>.csv       > profiles/<name>.md

`launches`: the csv of `ncu --metrics gpu__time_duration.sum --clock-control none --csv --log-file ...`: launches, total and mean
duration and share per kernel.  `raw`: the csv of `ncu -i <report> --page raw --csv` of a `--set full` capture: one column per
captured launch with the metrics the roofline discussion of DESIGN.md uses (duration, DRAM bytes, fp64 / DMMA pipe activity,
issue slots, occupancy, stall reasons).
"""
from __future__ import annotations

import collections
import csv
import re
import sys

RAW_METRICS = [
    ("duration", "gpu__time_duration.sum"),
    ("DRAM read", "dram__bytes_read.sum"),
    ("DRAM written", "dram__bytes_write.sum"),
    ("DRAM throughput % of peak", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"),
    ("L2 -> SM read bytes (lts__t_bytes, all)", "lts__t_bytes.sum"),
    ("fp64 tensor-path operations (DMMA flops)", "sm__ops_path_tensor_src_fp64.sum"),
    ("DMMA sub-pipe instructions, % of peak while active", "sm__inst_executed_pipe_tensor_subpipe_dmma.avg.pct_of_peak_sustained_active"),
    ("fp64 vector pipe (DFMA) cycles active %", "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
    ("issue slots busy %", "smsp__issue_active.avg.pct_of_peak_sustained_active"),
    ("achieved occupancy %", "sm__warps_active.avg.pct_of_peak_sustained_active"),
    ("registers / thread", "launch__registers_per_thread"),
    ("dynamic shared memory / CTA", "launch__shared_mem_per_block_dynamic"),
    ("stall barrier per issue", "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio"),
    ("stall long scoreboard per issue", "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio"),
    ("stall short scoreboard per issue", "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio"),
    ("stall wait per issue", "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio"),
    ("stall math pipe throttle per issue", "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio"),
    ("stall sleeping (nanosleep) per issue", "smsp__average_warps_issue_stalled_sleeping_per_issue_active.ratio"),
]


def short(name: str) -> str:
    m = re.search(r"(\w+_kernel|\w+)\s*\(", name)
    return m.group(1) if m else name.split("(")[0].split("::")[-1]


def launches(path: str) -> None:
    with open(path, newline="") as f:
        rows = [r for r in csv.reader(f) if r]
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    h = rows[hdr]
    ik, iv, iu = h.index("Kernel Name"), h.index("Metric Value"), h.index("Metric Unit")
    tot, cnt, order = collections.Counter(), collections.Counter(), []
    scale = {"ns": 1e-3, "us": 1.0, "usecond": 1.0, "nsecond": 1e-3, "ms": 1e3, "msecond": 1e3, "second": 1e6}
    for r in rows[hdr + 1:]:
        if len(r) <= iv:
            continue
        k = short(r[ik])
        if k not in tot:
            order.append(k)
        tot[k] += float(r[iv].replace(",", "")) * scale.get(r[iu], 1.0)
        cnt[k] += 1
    all_us = sum(tot.values())
    print("| kernel | launches | total us | mean us | share |")
    print("|---|---|---|---|---|")
    for k in sorted(order, key=lambda q: -tot[q]):
        print(f"| {k} | {cnt[k]} | {tot[k]:.0f} | {tot[k] / cnt[k]:.1f} | {100 * tot[k] / all_us:.2f} % |")
    print(f"| **all** | {sum(cnt.values())} | {all_us:.0f} | | 100 % |")


def raw(path: str) -> None:
    with open(path, newline="") as f:
        rows = [r for r in csv.reader(f) if r]
    h, units, data = rows[0], rows[1], rows[2:]
    ik = h.index("Kernel Name")
    print("| metric | unit | " + " | ".join(f"{short(r[ik])} #{n}" for n, r in enumerate(data)) + " |")
    print("|---|---|" + "---|" * len(data))
    for label, m in RAW_METRICS:
        if m not in h:
            continue
        j = h.index(m)
        print(f"| {label} (`{m}`) | {units[j]} | " + " | ".join(r[j] for r in data) + " |")


def main() -> None:
    if len(sys.argv) != 3 or sys.argv[1] not in ("launches", "raw"):
        sys.exit(__doc__)
    (launches if sys.argv[1] == "launches" else raw)(sys.argv[2])


if __name__ == "__main__":
    main()
