"""Summarise an Nsight Compute capture of the library's kernels as text and record its DRAM traffic.

    python -m paper_2606_20537_b200.ncu_summary REPORT.ncu-rep --name esc_scan_kernel_cold \
        --out profiles/r02_scan_w16_ncu_full.txt --command "<the ncu command that made the report>" [--launch 0]

reads the report with `ncu -i REPORT --page raw --csv` (works without a GPU), writes the selected counters of one
captured launch to --out (with the command, so the file names what made it), and stores that launch's
dram__bytes_read.sum / dram__bytes_write.sum under `name` in profiles/traffic.json together with the commit the
working tree was at.  bench.py reads roofline.traffic from that file, so a kernel change that is not re-captured
shows up as a stale commit there rather than as a silently wrong literal.
"""
import argparse
import csv
import io
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SELECTED = [
    "gpu__time_duration.sum", "launch__grid_size", "launch__block_size", "launch__cluster_size", "launch__registers_per_thread",
    "launch__shared_mem_per_block_dynamic", "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_registers",
    "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "lts__t_bytes.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__mem_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "sm__cycles_elapsed.max", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_membar_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_sleeping_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_lg_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio",
]

UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def read_raw(report):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    header, units = rows[0], rows[1]
    return header, units, rows[2:]


def git_commit():
    try:
        return subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], check=True, capture_output=True,
                              text=True).stdout.strip()
    except (OSError, subprocess.CalledProcessError):
        return "unknown"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--name", required=True, help="key in profiles/traffic.json (e.g. esc_copy_kernel, esc_scan_kernel_cold)")
    ap.add_argument("--out", required=True, help="text summary to write (under profiles/)")
    ap.add_argument("--command", required=True, help="the full ncu command that produced the report")
    ap.add_argument("--launch", type=int, default=0, help="which captured launch of the report to summarise")
    ap.add_argument("--title", default="")
    ap.add_argument("--note", default="")
    a = ap.parse_args()
    header, units, rows = read_raw(a.report)
    row = rows[a.launch]
    col = {h: i for i, h in enumerate(header)}
    kname = row[col["Kernel Name"]] if "Kernel Name" in col else "?"
    lines = []
    if a.title:
        lines.append(a.title)
    lines.append("Kernel: %s (launch %d of %d captured)" % (kname, a.launch, len(rows)))
    lines.append("Command (one B200 under gpurun, after the same command exited 0 without ncu):")
    lines.append("  " + a.command)
    lines.append("Read here with: ncu -i <report> --page raw --csv  (python -m paper_2606_20537_b200.ncu_summary; selected rows below)")
    if a.note:
        lines.append(a.note)
    lines.append("")
    vals = {}
    for m in SELECTED:
        if m in col:
            v, u = row[col[m]], units[col[m]]
            vals[m] = (v, u)
            lines.append("%-86s %s %s" % (m, v, u))

    def to_bytes(m):
        v, u = vals[m]
        return float(v.replace(",", "")) * UNIT_SCALE.get(u, 1.0)
    commit = git_commit()
    lines.append("")
    lines.append("working tree at commit %s when summarised" % commit)
    os.makedirs(os.path.dirname(os.path.abspath(a.out)), exist_ok=True)
    with open(a.out, "w") as f:
        f.write("\n".join(lines) + "\n")
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        d = json.load(open(tpath))
    except (OSError, ValueError):
        d = {"what": "per-launch DRAM bytes of the library's kernels from ncu --set full captures; written by "
                     "python -m paper_2606_20537_b200.ncu_summary, read by bench.py (roofline.traffic)", "kernels": {}}
    d["kernels"][a.name] = {"kernel": kname, "dram_read_bytes": to_bytes("dram__bytes_read.sum"),
                            "dram_write_bytes": to_bytes("dram__bytes_write.sum"),
                            "duration_us_under_ncu": vals.get("gpu__time_duration.sum", ("?", ""))[0],
                            "file": os.path.relpath(os.path.abspath(a.out), ROOT), "commit": commit, "command": a.command}
    with open(tpath, "w") as f:
        json.dump(d, f, indent=1, sort_keys=True)
        f.write("\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
