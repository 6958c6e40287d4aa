"""Summarise an `ncu --set full` report of the coarse-op kernels as text under profiles/.

    python -m paper_2212_12559_b200.ncu_summary REPORT.ncu-rep --out profiles/r02_ncu_full_c4.md \\
        --title "C4 ..." --command "<the full gpurun/ncu command that made the report>" \\
        [--config C4 --links i16 --path 2 --daggers 0,1 --csv profiles/r02_ncu_traffic.csv] [--reading "..."]

Writes a Markdown table (one column per captured launch) of the metrics the roofline discussion uses,
and - when --config is given - appends one row per launch to the traffic table that bench.py reads for
`roofline.traffic` (dram__bytes_read.sum + dram__bytes_write.sum per launch).  Needs the `ncu` CLI
(reading a report needs no GPU).
"""
from __future__ import annotations

import argparse
import csv
import io
import os
import subprocess

METRICS = [
    "gpu__time_duration.sum", "launch__grid_size", "launch__block_size", "launch__registers_per_thread",
    "launch__shared_mem_per_block_dynamic", "launch__cluster_dim_x", "launch__cluster_max_active", "dram__bytes_read.sum", "dram__bytes_write.sum",
    "dram__bytes_read.sum.per_second", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_tensor_subpipe_imma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
    "sm__cycles_elapsed.avg", "gpc__cycles_elapsed.avg.per_second",
]


def read_report(path: str):
    """`path`: an .ncu-rep file, or the text of `ncu -i REPORT --page raw --csv --print-units base` saved as .csv
    (reports of several captures exceed what gpurun brings back; the raw page is exported on the GPU box)."""
    if path.endswith(".csv"):
        with open(path) as f:
            out = f.read()
    else:
        out = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv", "--print-units", "base"],
                             capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    return hdr, units, data


def short_kernel(name: str) -> str:
    name = name.replace("void ", "").replace("coarse::", "")
    return name.split("(")[0] if "(" in name and name.index("(") > name.find(">") else name


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--out", required=True)
    ap.add_argument("--title", default="")
    ap.add_argument("--command", required=True, help="the full command that produced the report")
    ap.add_argument("--reading", default="", help="free text appended under 'Reading'")
    ap.add_argument("--config", default="")
    ap.add_argument("--links", default="c64")
    ap.add_argument("--path", type=int, default=0)
    ap.add_argument("--daggers", default="", help="dagger of each captured launch, in order, e.g. 0,1")
    ap.add_argument("--csv", default="")
    args = ap.parse_args()

    hdr, units, data = read_report(args.report)
    kn = hdr.index("Kernel Name")
    cols = ["`" + short_kernel(r[kn]) + "`" for r in data]
    lines = ["# " + (args.title or os.path.basename(args.report)), "", "Command (run on the B200 box through gpurun; the report was read here with `ncu -i`):",
             "", "    " + args.command, "", "| metric | unit | " + " | ".join(cols) + " |", "|---|---|" + "---|" * len(cols)]
    vals = {}
    for m in METRICS:
        if m not in hdr:
            continue
        i = hdr.index(m)
        vals[m] = [r[i] for r in data]
        lines.append(f"| {m} | {units[i]} | " + " | ".join(vals[m]) + " |")
    rd = [int(float(x.replace(",", ""))) for x in vals["dram__bytes_read.sum"]]
    wr = [int(float(x.replace(",", ""))) for x in vals["dram__bytes_write.sum"]]
    lines.append("| **traffic = dram read + write** | byte | " + " | ".join(f"**{a + b}**" for a, b in zip(rd, wr)) + " |")
    if args.reading:
        lines += ["", "## Reading", "", args.reading]
    with open(args.out, "w") as f:
        f.write("\n".join(lines) + "\n")
    if args.config and args.csv:
        daggers = [int(x) for x in args.daggers.split(",")] if args.daggers else list(range(len(data)))
        new = not os.path.exists(args.csv)
        with open(args.csv, "a", newline="") as f:
            w = csv.writer(f)
            if new:
                w.writerow(["config", "links", "path", "dagger", "kernel", "time_ns", "dram_bytes_read", "dram_bytes_write", "summary"])
            for k, r in enumerate(data):
                t = vals["gpu__time_duration.sum"][k].replace(",", "")
                w.writerow([args.config, args.links, args.path, daggers[k], short_kernel(r[kn]), int(float(t)), rd[k], wr[k],
                            os.path.basename(args.out)])
    print(args.out)


if __name__ == "__main__":
    main()
