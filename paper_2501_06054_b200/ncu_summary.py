"""Text summary of an Nsight Compute report of the trace kernels (what profiles/r*_ncu_*.md hold).

    python -m paper_2501_06054_b200.ncu_summary report.ncu-rep [launch_index ...]

Prints one markdown table per selected launch (default: all) with the metrics the roofline discussion of
DESIGN.md section 7 uses, and the warp-state sample shares of the source page.  Needs `ncu` on PATH; reads the
report only (no GPU)."""
from __future__ import annotations

import csv
import subprocess
import sys

METRICS = [
    ("kernel duration", "gpu__time_duration.sum"),
    ("SM cycles elapsed", "sm__cycles_elapsed.avg"),
    ("grid", "launch__grid_size"), ("block", "launch__block_size"),
    ("registers/thread", "launch__registers_per_thread"),
    ("dynamic smem/block", "launch__shared_mem_per_block_dynamic"),
    ("achieved occupancy %", "sm__warps_active.avg.pct_of_peak_sustained_active"),
    ("warp instructions executed", "smsp__inst_executed.sum"),
    ("active threads per warp instruction (32 = no divergence)", "smsp__thread_inst_executed_per_inst_executed.ratio"),
    ("issue slots busy % (1 warp-instr/clk/SMSP = 100)", "smsp__issue_active.avg.pct_of_peak_sustained_active"),
    ("eligible warps per cycle per SMSP", "smsp__warps_eligible.avg.per_cycle_active"),
    ("FMA-heavy pipe busy % of elapsed cycles (integer multiplier)", "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed"),
    ("FMA pipe (heavy + lite) busy %", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_elapsed"),
    ("FMA-lite instructions %", "sm__inst_executed_pipe_fmalite.avg.pct_of_peak_sustained_active"),
    ("ALU (logic) pipe busy %", "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_elapsed"),
    ("FP64 pipe busy %", "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed"),
    ("FP64 warp instructions", "smsp__inst_executed_pipe_fp64.sum"),
    ("XU pipe (MUFU/POPC/conversions) %", "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_elapsed"),
    ("LSU pipe %", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_elapsed"),
    ("tensor pipe %", "sm__inst_executed_pipe_tensor_subpipe_hmma.avg.pct_of_peak_sustained_active"),
    ("local-memory (spill) load requests", "l1tex__t_requests_pipe_lsu_mem_local_op_ld.sum"),
    ("DRAM bytes read", "dram__bytes_read.sum"), ("DRAM bytes written", "dram__bytes_write.sum"),
    ("DRAM throughput % of peak", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"),
]


def main(argv):
    rep = argv[1]
    pick = [int(a) for a in argv[2:]]
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr, units = rows[0], rows[1]
    ikernel = hdr.index("Kernel Name")
    for li, vals in enumerate(rows[2:]):
        if pick and li not in pick:
            continue
        d = dict(zip(hdr, vals))
        u = dict(zip(hdr, units))
        print(f"### launch {li}: `{vals[ikernel]}`\n")
        print("| metric | value | unit |\n|---|---|---|")
        for label, key in METRICS:
            if key in d:
                print(f"| {label} (`{key}`) | {d[key]} | {u[key]} |")
        stalls = {k.split("issue_stalled_")[1].split("_per_issue")[0]: float(v) for k, v in d.items()
                  if "issue_stalled" in k and k.endswith("per_issue_active.ratio") and v}
        tot = sum(stalls.values())
        if tot > 0:
            top = sorted(stalls.items(), key=lambda kv: -kv[1])[:9]
            print("\nWarp states (share of warp-cycles, `smsp__average_warps_issue_stalled_*`): " +
                  ", ".join(f"{k} {100 * v / tot:.1f} %" for k, v in top) + "\n")


if __name__ == "__main__":
    main(sys.argv)
