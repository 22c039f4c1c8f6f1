"""Turn an Nsight Compute report into the text summaries kept under profiles/.

    python -m paper_2009_00735_b200.ncu_summary REPORT.ncu-rep --name r2_k_signature_mma_cfg4 \
        --kernel k_signature_mma --config 4 --command "<the full ncu command that wrote the report>"

writes profiles/<name>.md (the metrics that matter for the roofline of this path, one table per captured launch) and
merges the per-launch constants bench.py cites (DRAM bytes, shared-memory wavefronts) into
profiles/r2_ncu_constants.json under [kernel][config].  Reads the report with `ncu -i ... --page raw --csv`; nothing here
runs on the GPU.
"""
from __future__ import annotations
import argparse
import csv
import io
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
WANTED = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
    "sm__cycles_active.avg", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "l1tex__data_pipe_lsu_wavefronts.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_atom.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_ld.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_st.sum",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_atom.sum",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_ld.sum",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_st.sum",
    "smsp__inst_executed_op_shared_atom.sum", "smsp__sass_inst_executed_op_shared_ld.sum",
    "smsp__sass_inst_executed_op_shared_st.sum",
    "lts__t_bytes.sum", "l1tex__t_bytes_pipe_lsu_mem_global_op_ld.sum",
    "launch__grid_size", "launch__block_size", "launch__registers_per_thread",
    "launch__shared_mem_per_block_dynamic", "sm__warps_active.avg.pct_of_peak_sustained_active",
]
STALL_PREFIX = "smsp__average_warps_issue_stalled_"


def read_report(path):
    out = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    # first row: column names, second row: units, then one row per captured launch
    names, units = rows[0], rows[1]
    return names, units, rows[2:]


def to_float(v):
    try:
        return float(v.replace(",", ""))
    except ValueError:
        return None


UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--name", required=True, help="basename of the summary under profiles/")
    ap.add_argument("--kernel", required=True, help="kernel the constants belong to, e.g. k_signature_mma")
    ap.add_argument("--config", required=True, help="BASELINE.json config number the capture ran on")
    ap.add_argument("--command", required=True, help="the full command that produced the report")
    ap.add_argument("--note", default="")
    ap.add_argument("--points", type=int, default=0, help="material points of the captured launch (0 = the whole config)")
    args = ap.parse_args()
    names, units, launches = read_report(args.report)
    col = {n: i for i, n in enumerate(names)}
    lines = [f"# ncu --set full summary: `{args.kernel}` on config {args.config}", "",
             "Command (under gpurun, one B200, after the same command had exited 0 without ncu):", "",
             f"    {args.command}", ""]
    if args.note:
        lines += [args.note, ""]
    consts = None
    for li, row in enumerate(launches):
        kname = row[col["Kernel Name"]] if "Kernel Name" in col else "?"
        lines += [f"## launch {li}: `{kname}`", "", "| metric | unit | value |", "|---|---|---|"]
        picked = [n for n in WANTED if n in col] + sorted(n for n in names if n.startswith(STALL_PREFIX) and n.endswith("_per_issue_active.ratio"))
        for n in picked:
            lines.append(f"| `{n}` | {units[col[n]]} | {row[col[n]]} |")
        lines.append("")
        if args.kernel in kname and consts is None:
            def val(n):
                if n not in col:
                    return None
                v = to_float(row[col[n]])
                return None if v is None else v * UNIT_SCALE.get(units[col[n]], 1.0)
            rd, wr = val("dram__bytes_read.sum"), val("dram__bytes_write.sum")
            consts = {"dram_bytes": (rd or 0.0) + (wr or 0.0),
                      "lsu_wavefronts_shared": val("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"),
                      "lsu_wavefronts_shared_atom": val("l1tex__data_pipe_lsu_wavefronts_mem_shared_op_atom.sum"),
                      "inst_executed": val("smsp__inst_executed.sum"),
                      "points": args.points,
                      "capture": f"profiles/{args.name}.md"}
    os.makedirs(os.path.join(ROOT, "profiles"), exist_ok=True)
    with open(os.path.join(ROOT, "profiles", args.name + ".md"), "w") as f:
        f.write("\n".join(lines))
    if consts:
        path = os.path.join(ROOT, "profiles", "r2_ncu_constants.json")
        allc = json.load(open(path)) if os.path.exists(path) else {}
        allc.setdefault(args.kernel, {})[str(args.config)] = consts
        with open(path, "w") as f:
            json.dump(allc, f, indent=1, sort_keys=True)
    print("\n".join(lines[:12]))


if __name__ == "__main__":
    main()
