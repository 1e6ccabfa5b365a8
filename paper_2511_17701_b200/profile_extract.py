"""Text extracts of an Nsight Compute report for profiles/ (run where ncu is installed; no GPU needed).

    python -m paper_2511_17701_b200.profile_extract <report.ncu-rep> <kernel-name-substring> <particles-per-launch> <out-prefix>

Writes, for the first launch in the report whose kernel name contains the substring:
    <out-prefix>.csv          key,value rows that bench.py reads (kernel, particles_per_launch, dram__bytes_*.sum,
                              flop_executed_per_launch, warp_inst_per_32_particles) plus the headline counters
    <out-prefix>_raw.csv      the full `ncu --page raw --csv` row of that launch (every metric of --set full), transposed
    <out-prefix>_opcodes.csv  executed warp / thread instructions per SASS opcode (from `--page source --print-source sass`)
"""
from __future__ import annotations

import collections
import csv
import subprocess
import sys

KEYS = ["gpu__time_duration.sum", "smsp__inst_executed.sum", "smsp__issue_active.avg.pct_of_peak_sustained_active",
        "launch__registers_per_thread", "launch__grid_size", "launch__block_size", "launch__occupancy_limit_registers",
        "launch__occupancy_limit_shared_mem", "sm__warps_active.avg.pct_of_peak_sustained_active",
        "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
        "lts__throughput.avg.pct_of_peak_sustained_elapsed", "l1tex__throughput.avg.pct_of_peak_sustained_elapsed",
        "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "smsp__thread_inst_executed_per_inst_executed.ratio",
        "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
        "smsp__inst_executed_op_shared_atom.sum"]
FLOP = {"FFMA": 2, "FMUL": 1, "FADD": 1, "DFMA": 2, "DMUL": 1, "DADD": 1}


def _ncu(rep, *args):
    return subprocess.run(["ncu", "-i", rep, *args], capture_output=True, text=True, check=True).stdout


def main():
    rep, sub, particles, prefix = sys.argv[1], sys.argv[2], float(sys.argv[3]), sys.argv[4]
    rows = list(csv.reader(_ncu(rep, "--page", "raw", "--csv").splitlines()))
    hdr, units = rows[0], rows[1]
    ik = hdr.index("Kernel Name")
    row = next(r for r in rows[2:] if sub in r[ik])
    val = dict(zip(hdr, row))
    num = lambda k: float(val[k].replace(",", ""))
    with open(prefix + "_raw.csv", "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["metric", "unit", "value"])
        for h, u, v in zip(hdr, units, row):
            w.writerow([h, u, v])
    # opcode histogram of the same kernel
    src = list(csv.reader(_ncu(rep, "--page", "source", "--csv", "--print-source", "sass").splitlines()))
    ops_w, ops_t = collections.Counter(), collections.Counter()
    take, cols = False, None
    for r in src:
        if r and r[0] == "Kernel Name":
            if take:
                break
            take = sub in r[1]
            cols = None
            continue
        if not take or not r:
            continue
        if r[0] == "Address":
            cols = (r.index("Source"), r.index("Instructions Executed"), r.index("Thread Instructions Executed"))
            continue
        if cols is None:
            continue
        t = r[cols[0]].split()
        if not t:
            continue
        op = (t[1] if t[0].startswith("@") else t[0]).split(".")[0]
        try:
            ops_w[op] += int(r[cols[1]]); ops_t[op] += int(r[cols[2]])
        except ValueError:
            pass
    with open(prefix + "_opcodes.csv", "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["opcode", "warp_instructions", "thread_instructions", "warp_instructions_per_32_particles"])
        for op, n in ops_w.most_common():
            w.writerow([op, n, ops_t[op], f"{n / (particles / 32):.2f}"])
    flop = sum(FLOP[o] * ops_t[o] for o in FLOP)
    with open(prefix + ".csv", "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["# key", "value   (first launch of the kernel in " + rep.split("/")[-1] + ")"])
        w.writerow(["kernel", val["Kernel Name"].split("(")[0]])
        w.writerow(["particles_per_launch", f"{particles:.0f}"])
        w.writerow(["flop_executed_per_launch", flop])
        w.writerow(["warp_inst_per_32_particles", f"{num('smsp__inst_executed.sum') / (particles / 32):.1f}"])
        unit = dict(zip(hdr, units))
        scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}
        for k in KEYS:
            if k in val:
                v = val[k].replace(",", "")
                if unit[k] in scale:                  # bytes in plain bytes whatever unit ncu chose to print
                    v = f"{float(v) * scale[unit[k]]:.0f}"
                w.writerow([k, v, "byte" if unit[k] in scale else unit[k]])
        for h in hdr:
            if h.startswith("smsp__average_warps_issue_stalled") and h.endswith("per_issue_active.ratio") and val[h] not in ("0", ""):
                w.writerow([h, val[h]])
    print("wrote", prefix + ".csv", prefix + "_raw.csv", prefix + "_opcodes.csv", "flop/particle", flop / particles)


if __name__ == "__main__":
    main()
