"""Summarise an `ncu --set full` report of the marcher: a markdown table for profiles/ and the per-launch
counters bench.py reads (profiles/r2_counters.json: DRAM bytes, warp instructions, duration per launch).

  python -m paper_1012_2909_b200.ncu_counters --rep gpurun_out/c3_ea.ncu-rep --workload C3 --mode ea --tf src \
      --frames 0,180 --cmd "<the profiled command>" --title "..." --md profiles/r2_c3_ea_full.md

Runs here (no GPU needed): `ncu -i <rep> --page raw --csv` is the only tool called.  bench.py never types
these numbers in: it looks them up by (workload, mode, table, kernel) and prints null where no capture exists.
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEEP = ["gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "dram__bytes_read.sum.per_second",
        "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
        "l1tex__t_sector_hit_rate.pct", "lts__t_sector_hit_rate.pct",
        "l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum", "l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum",
        "lts__t_sectors_srcunit_tex_op_read.sum", "lts__t_sectors_srcunit_tex_op_read_lookup_miss.sum",
        "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
        "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
        "sm__throughput.avg.pct_of_peak_sustained_elapsed", "smsp__issue_active.avg.pct_of_peak_sustained_active",
        "smsp__inst_executed.sum", "smsp__thread_inst_executed_per_inst_executed.ratio",
        "sm__inst_executed_pipe_lsu.sum", "sm__inst_executed_pipe_fma.sum", "sm__inst_executed_pipe_alu.sum",
        "sm__warps_active.avg.pct_of_peak_sustained_active", "launch__registers_per_thread", "launch__shared_mem_per_block",
        "launch__grid_size", "launch__block_size", "launch__waves_per_multiprocessor", "launch__occupancy_limit_registers",
        "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_warps", "sm__cycles_elapsed.max",
        "smsp__warps_eligible.avg.per_cycle_active"]
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
        "ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6, "second": 1e6, "usecond": 1.0, "msecond": 1e3, "nsecond": 1e-3}


def raw_rows(rep):
    txt = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(txt)))
    start = next(i for i, r in enumerate(rows) if r and r[0] == "ID")
    return rows[start], rows[start + 1], rows[start + 2:]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rep", required=True)
    ap.add_argument("--workload", required=True)
    ap.add_argument("--mode", required=True, choices=["ea", "mip"])
    ap.add_argument("--tf", default="src")
    ap.add_argument("--frames", default="")
    ap.add_argument("--kernel", default=None, help="kernel function name to keep (default: every captured launch)")
    ap.add_argument("--cmd", required=True)
    ap.add_argument("--title", required=True)
    ap.add_argument("--md", required=True)
    ap.add_argument("--json", default=os.path.join(ROOT, "profiles", "r2_counters.json"))
    ap.add_argument("--no-json", action="store_true")
    a = ap.parse_args()
    hdr, units, rows = raw_rows(a.rep)
    kn = hdr.index("Kernel Name")
    if a.kernel:
        rows = [r for r in rows if a.kernel in r[kn]]
    n = len(rows)
    lines = [f"# {a.title}", "", "Command (under gpurun, one B200, after the same command exited 0 without ncu):", "", f"    {a.cmd}", "",
             "Read back with `python -m paper_1012_2909_b200.ncu_counters` (`ncu -i <report> --page raw --csv`); selected metrics per captured launch:", "",
             "| metric | unit | " + " | ".join(f"launch {i + 1}" for i in range(n)) + " |", "|---|---|" + "---|" * n,
             "| kernel | | " + " | ".join(r[kn].replace("|", "\\|")[:70] for r in rows) + " |"]
    for h in KEEP:
        if h in hdr:
            i = hdr.index(h)
            lines.append(f"| {h} | {units[i]} | " + " | ".join(r[i] for r in rows) + " |")
    lines += ["", "Warp stall reasons (warps stalled per issue-active cycle, `smsp__average_warps_issue_stalled_*_per_issue_active.ratio`):", "",
              "| reason | " + " | ".join(f"launch {i + 1}" for i in range(n)) + " |", "|---|" + "---|" * n]
    pre, post = "smsp__average_warps_issue_stalled_", "_per_issue_active.ratio"
    for i, h in enumerate(hdr):
        if h.startswith(pre) and h.endswith(post) and "not_issued" not in h:
            vals = [r[i] for r in rows]
            try:
                if max(float(v) for v in vals) < 0.02:
                    continue
            except ValueError:
                continue
            lines.append(f"| {h[len(pre):-len(post)]} | " + " | ".join(vals) + " |")
    with open(a.md, "w") as f:
        f.write("\n".join(lines) + "\n")
    print(a.md)
    if a.no_json or not rows:
        return

    def val(r, name):
        i = hdr.index(name)
        return float(r[i].replace(",", "")) * UNIT.get(units[i], 1.0)

    commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    kernels = sorted({r[kn].split("(")[0].split("::")[-1].split("<")[0].strip() for r in rows})
    cap = {"workload": a.workload, "mode": a.mode, "tf": a.tf, "kernel": kernels[0] if len(kernels) == 1 else ",".join(kernels),
           "frames": [int(v) for v in a.frames.split(",") if v != ""],
           "dram_bytes": [val(r, "dram__bytes_read.sum") + val(r, "dram__bytes_write.sum") for r in rows],
           "warp_instructions": [val(r, "smsp__inst_executed.sum") for r in rows],
           "duration_us": [val(r, "gpu__time_duration.sum") for r in rows],
           "source": os.path.relpath(a.md, ROOT), "commit": commit, "command": a.cmd}
    doc = {"captures": []}
    if os.path.exists(a.json):
        with open(a.json) as f:
            doc = json.load(f)
    doc["captures"] = [c for c in doc["captures"]
                       if not (c["workload"] == cap["workload"] and c["mode"] == cap["mode"] and c.get("tf") == cap["tf"] and c["kernel"] == cap["kernel"])]
    doc["captures"].append(cap)
    with open(a.json, "w") as f:
        json.dump(doc, f, indent=1)
        f.write("\n")
    print(a.json)


if __name__ == "__main__":
    main()
