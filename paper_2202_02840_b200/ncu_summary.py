"""Text summaries of an Nsight Compute capture of libcrk's kernels.

    python -m paper_2202_02840_b200.ncu_summary --rep gpurun_out/prof.ncu-rep --workload "cosmo n_side=256" \
        --json profiles/r02_ncu_kernels.json --md profiles/r02_ncu_kernels.md --command "<the ncu command line>"

Reads `ncu -i <rep> --page raw --csv` (or a CSV made that way, --csv) and writes, per kernel, the metrics the roofline
discussion uses: duration, DRAM bytes, FMA-pipe / issue utilisation, instruction count, shared-memory wavefronts and bank
conflicts, registers, occupancy and the stall reasons per issue.  bench.py reads the JSON for `roofline.traffic` (only for
the workload named in it).  Nothing here runs on the GPU.
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import subprocess

METRICS = {
    "gpu__time_duration.sum": "time_ms",
    "dram__bytes_read.sum": "dram_bytes_read",
    "dram__bytes_write.sum": "dram_bytes_write",
    "launch__registers_per_thread": "registers",
    "sm__warps_active.avg.pct_of_peak_sustained_active": "warps_active_pct",
    "smsp__issue_active.avg.pct_of_peak_sustained_active": "issue_active_pct",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active": "fma_pipe_pct",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active": "alu_pipe_pct",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active": "lsu_pipe_pct",
    "smsp__inst_executed.sum": "warp_instructions",
    "smsp__thread_inst_executed_per_inst_executed.ratio": "active_lanes_per_instruction",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum": "shared_wavefronts",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum": "shared_bank_conflicts",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed": "l1tex_throughput_pct",
    "lts__throughput.avg.pct_of_peak_sustained_elapsed": "l2_throughput_pct",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed": "dram_throughput_pct",
}
STALLS = ("long_scoreboard", "short_scoreboard", "barrier", "wait", "mio_throttle", "math_pipe_throttle", "not_selected",
          "lg_throttle", "branch_resolving", "dispatch_stall", "no_instruction")
UNIT_SCALE = {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3, "byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def short_name(full: str) -> str:
    """k_forces<false>(SweepArgs) from the demangled name ncu prints"""
    n = full.replace("(anonymous namespace)::", "").replace("<unnamed>::", "").replace("void ", "")
    n = n.split("(")[0].strip()
    return n or full


def read_raw(rep: str | None, csv_path: str | None):
    if csv_path:
        text = open(csv_path).read()
    else:
        text = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(text)))
    while rows and "Kernel Name" not in rows[0]:
        rows.pop(0)
    hdr, units, data = rows[0], rows[1], rows[2:]
    return hdr, units, data


def summarise(hdr, units, data):
    col = {h: i for i, h in enumerate(hdr)}
    out = {}
    for r in data:
        name = short_name(r[col["Kernel Name"]])
        k = {}
        for m, key in METRICS.items():
            if m not in col or r[col[m]] == "":
                continue
            v = float(r[col[m]].replace(",", ""))
            u = units[col[m]]
            if key == "time_ms" or key.startswith("dram_bytes"):
                v *= UNIT_SCALE.get(u, 1.0)
            k[key] = v
        for st in STALLS:
            m = f"smsp__average_warps_issue_stalled_{st}_per_issue_active.ratio"
            if m in col and r[col[m]] != "":
                k.setdefault("stalls_per_issue", {})[st] = float(r[col[m]])
        base = name.split("<")[0]
        out.setdefault(base if base not in out else name, k)       # first launch of each kernel (template variants share a row)
    return out


def to_md(kernels, workload, command):
    keys = ["time_ms", "registers", "warps_active_pct", "issue_active_pct", "fma_pipe_pct", "alu_pipe_pct", "lsu_pipe_pct",
            "warp_instructions", "active_lanes_per_instruction", "dram_bytes_read", "dram_bytes_write", "shared_wavefronts",
            "shared_bank_conflicts", "l1tex_throughput_pct", "l2_throughput_pct", "dram_throughput_pct"]
    names = list(kernels)
    lines = [f"# ncu --set full summary, workload: {workload}", "", "Command:", "", "```", command, "```", "",
             "| metric | " + " | ".join(names) + " |", "|---|" + "---|" * len(names)]
    for k in keys:
        lines.append(f"| {k} | " + " | ".join(f"{kernels[n].get(k, float('nan')):.4g}" for n in names) + " |")
    for st in STALLS:
        lines.append(f"| stall {st} / issue | " + " | ".join(f"{kernels[n].get('stalls_per_issue', {}).get(st, float('nan')):.3g}" for n in names) + " |")
    return "\n".join(lines) + "\n"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rep")
    ap.add_argument("--csv")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--json", required=True)
    ap.add_argument("--md")
    ap.add_argument("--command", default="(not recorded)")
    a = ap.parse_args()
    hdr, units, data = read_raw(a.rep, a.csv)
    kernels = summarise(hdr, units, data)
    with open(a.json, "w") as f:
        json.dump({"workload": a.workload, "source": a.rep or a.csv, "command": a.command, "kernels": kernels}, f, indent=1)
    if a.md:
        with open(a.md, "w") as f:
            f.write(to_md(kernels, a.workload, a.command))


if __name__ == "__main__":
    main()
