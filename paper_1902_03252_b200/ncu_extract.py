"""Turns `ncu -i <report> --page raw --csv --print-units base` into what this repository keeps from a capture:

  * an entry of profiles/ncu_traffic.json -- dram__bytes_read.sum / dram__bytes_write.sum per launch of a mode's dominant
    kernel on a named workload, with the commit the capture was taken at (bench.py reports it as `roofline.traffic`);
  * a markdown table of the counters SURVEY 8(d) asks for (pipe utilisations, issue slots, registers, stalls).

    ncu -i prof.ncu-rep --page raw --csv --print-units base | \\
        python -m paper_1902_03252_b200.ncu_extract --kernel lt_grad_f64_kernel --workload cfg3_4096x4096_1000 \\
               --mode fp64 --commit $(git rev-parse --short HEAD) --json profiles/ncu_traffic.json --md -

Reads the CSV from stdin.  With several launches of the kernel in the report the longest one is taken (the main launch
of a wave-split grid).  No GPU needed: it only reads ncu's export.
"""
import argparse
import csv
import json
import os
import sys

COUNTERS = [
    "gpu__time_duration.sum",
    "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_uniform.avg.pct_of_peak_sustained_active",
    "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active",
    "smsp__warps_eligible.avg.per_cycle_active",
    "launch__registers_per_thread",
    "launch__occupancy_limit_registers",
    "launch__grid_size",
    "smsp__inst_executed.sum",
    "sm__cycles_active.avg",
    "sm__cycles_elapsed.avg.per_second",
    "dram__bytes_read.sum",
    "dram__bytes_write.sum",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_ffma_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_fadd_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_fmul_pred_on.sum",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_dispatch_stall_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
]


def read_rows(stream):
    rows = [r for r in csv.reader(stream) if r]
    while rows and "Kernel Name" not in rows[0]:        # ncu may print ==PROF== lines first
        rows.pop(0)
    if len(rows) < 3:
        raise SystemExit("no ncu raw page on stdin")
    hdr, units = rows[0], rows[1]
    return hdr, units, rows[2:]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kernel", required=True, help="substring of the kernel name")
    ap.add_argument("--workload", help="workload name as bench.py prints it (config.workload)")
    ap.add_argument("--mode", help="fp64 | fp32 | mixed")
    ap.add_argument("--commit", default=None)
    ap.add_argument("--command", default=None, help="the ncu command that made the report (kept in the JSON)")
    ap.add_argument("--json", default=None, help="profiles/ncu_traffic.json to update")
    ap.add_argument("--md", default=None, help="file to append the counter table to ('-' = stdout)")
    ap.add_argument("--sum", action="store_true",
                    help="the report holds the launches of ONE step (a catalogue beyond one constant-bank slot-load runs "
                         "as several launches that carry partial sums): the JSON entry sums bytes and durations over them")
    a = ap.parse_args()
    hdr, units, rows = read_rows(sys.stdin)
    col = {h: i for i, h in enumerate(hdr)}
    cand = [r for r in rows if a.kernel in r[col["Kernel Name"]]]
    if not cand:
        raise SystemExit("kernel %r not in the report" % a.kernel)

    def num(r, name):
        try:
            return float(r[col[name]].replace(",", ""))
        except (KeyError, ValueError):
            return None
    row = max(cand, key=lambda r: num(r, "gpu__time_duration.sum") or 0.0)
    if a.json:
        if not (a.workload and a.mode):
            raise SystemExit("--json needs --workload and --mode")
        rec = json.load(open(a.json)) if os.path.exists(a.json) else {"captures": {}}
        rec.setdefault("what", "dram__bytes_read.sum / dram__bytes_write.sum (bytes) per launch of each mode's dominant kernel, "
                               "from `ncu --set full` captures; written by paper_1902_03252_b200/ncu_extract.py")
        rec["commit"] = a.commit or rec.get("commit")
        over = cand if a.sum else [row]

        def tot(name):
            return sum(num(r, name) or 0.0 for r in over)
        rec["captures"]["%s/%s" % (a.workload, a.mode)] = {
            "kernel": row[col["Kernel Name"]].split("(")[0].strip(), "launches_in_report": len(cand),
            "launches_summed": len(over),
            "dram_bytes_read": tot("dram__bytes_read.sum"), "dram_bytes_write": tot("dram__bytes_write.sum"),
            "duration_ns_under_ncu": tot("gpu__time_duration.sum"), "commit": a.commit, "command": a.command}
        json.dump(rec, open(a.json, "w"), indent=1, sort_keys=True)
    if a.md:
        out = sys.stdout if a.md == "-" else open(a.md, "a")
        out.write("\n### `%s`%s\n\n| metric | unit | value |\n|---|---|---|\n" % (
            row[col["Kernel Name"]].split("(")[0].strip(), " (%s, %s)" % (a.workload, a.mode) if a.workload else ""))
        for c in COUNTERS:
            if c in col:
                out.write("| `%s` | %s | %s |\n" % (c, units[col[c]], row[col[c]]))
        if out is not sys.stdout:
            out.close()


if __name__ == "__main__":
    main()
