"""Turns an `ncu --set full` report into the text summaries kept under profiles/.

    python -m paper_1811_06965_b200.ncu_summary REPORT.ncu-rep --md profiles/NAME.md [--title "..."]
                                                [--command "the command the capture was taken with"]
                                                [--traffic-key KEY]     # e.g. gemm_tcgen05:ffn1_fwd

Reads the report here (no GPU needed: `ncu -i REPORT --page raw --csv`), writes a markdown table of the
metrics the roofline argument uses (duration, DRAM bytes, L2 -> SM bytes, tensor-pipe activity, registers,
shared memory) with one column per captured launch, and - with --traffic-key - records the mean
`dram__bytes_read.sum + dram__bytes_write.sum` per launch under that key in profiles/ncu_traffic.json,
which is where bench.py takes `roofline.traffic` from.  profiles/ holds text only; this tool lives with
the package.
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

METRICS = [
    "gpu__time_duration.sum", "launch__grid_size", "launch__block_size", "launch__registers_per_thread",
    "launch__shared_mem_per_block_dynamic", "launch__cluster_dim_x", "sm__cycles_elapsed.avg", "sm__cycles_elapsed.avg.per_second",
    "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__mem_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__pipe_tensor_subpipe_hmma_cycles_active.avg.pct_of_peak_sustained_active",
    "l1tex__m_xbar2l1tex_read_bytes.sum", "l1tex__m_xbar2l1tex_read_bytes.sum.per_second",
    "lts__t_sector_hit_rate.pct", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__issue_active.avg.pct_of_peak_sustained_elapsed", "smsp__inst_executed.sum",
    "sm__pipe_xu_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "smsp__warp_issue_stalled_long_scoreboard_per_warp_active.pct",
]

_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def read_raw(report):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True)
    if out.returncode != 0:
        raise SystemExit("ncu failed: %s" % out.stderr[-2000:])
    rows = [r for r in csv.reader(io.StringIO(out.stdout)) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    return rows[start], rows[start + 1], rows[start + 2:]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--md", required=True)
    ap.add_argument("--title", default=None)
    ap.add_argument("--command", default=None)
    ap.add_argument("--traffic-key", default=None)
    ap.add_argument("--kernel", default=None, help="substring filter on the kernel name")
    ap.add_argument("--note", action="append", default=[])
    args = ap.parse_args()
    hdr, units, data = read_raw(args.report)
    idx = {h: i for i, h in enumerate(hdr)}
    if args.kernel:
        data = [d for d in data if args.kernel in d[idx["Kernel Name"]]]
    if not data:
        raise SystemExit("no launches in the report match")
    lines = ["# %s" % (args.title or os.path.basename(args.report)), ""]
    if args.command:
        lines += ["Command (one B200, via gpurun; the same command exited 0 without ncu first):", "", "    " + args.command, ""]
    lines += ["read here with `python -m paper_1811_06965_b200.ncu_summary %s ...` (= `ncu -i ... --page raw --csv`)." %
              os.path.basename(args.report), ""]
    lines.append("| metric | unit | " + " | ".join("launch %d" % i for i in range(len(data))) + " |")
    lines.append("|---|---|" + "---|" * len(data))
    lines.append("| `Kernel Name` |  | " + " | ".join(d[idx["Kernel Name"]].split("(")[0][-40:] for d in data) + " |")
    for m in METRICS:
        if m in idx:
            lines.append("| `%s` | %s | %s |" % (m, units[idx[m]], " | ".join(d[idx[m]] for d in data)))
    for n in args.note:
        lines += ["", n]
    os.makedirs(os.path.dirname(os.path.abspath(args.md)), exist_ok=True)
    with open(args.md, "w") as f:
        f.write("\n".join(lines) + "\n")
    if args.traffic_key:
        tot = []
        for d in data:
            b = 0.0
            for m in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                b += float(d[idx[m]].replace(",", "")) * _SCALE[units[idx[m]]]
            tot.append(b)
        p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
        j = json.load(open(p)) if os.path.exists(p) else {}
        j[args.traffic_key] = {"dram_bytes_per_launch": sum(tot) / len(tot), "launches": len(tot),
                               "source": os.path.relpath(os.path.abspath(args.md), ROOT),
                               "kernel": data[0][idx["Kernel Name"]].split("(")[0][-60:]}
        with open(p, "w") as f:
            json.dump(j, f, indent=1, sort_keys=True)
            f.write("\n")
    print("wrote", args.md)


if __name__ == "__main__":
    sys.exit(main())
