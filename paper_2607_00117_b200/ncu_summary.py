"""Reduce an Nsight Compute report to the text summaries kept under profiles/ and to the per-kernel operation counts that
bench.py's roofline uses (profiles/kernel_counts.json).

    python -m paper_2607_00117_b200.ncu_summary REPORT.ncu-rep --name r2x_cfg2_f64 --md "command that made the report" \
        [--counts KEY --work ORBIT_STEPS]

writes profiles/<name>_ncu_full_summary.csv (one column per profiled launch, the metrics listed in METRICS) and, with
--counts, stores under KEY (e.g. "integrate_kernel/barred/f64") the floating-point instructions the kernel EXECUTED per
thread and orbit-step (smsp__sass_thread_inst_executed_op_*_pred_on.sum.per_cycle_elapsed x sm__cycles_elapsed.avg of the first
profiled launch of that kernel / --work, the orbit-steps that launch integrated), its DRAM bytes per launch, and a hash of the kernel sources the report was taken from.
tests/test_library_host.py fails when that hash no longer matches csrc/: a roofline computed from stale counts is wrong.
Needs `ncu` on PATH (reads the report; no GPU).  Nothing here runs on the product path.
"""
import argparse
import csv
import hashlib
import io
import json
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
PROFILES = os.path.join(ROOT, "profiles")
COUNTS = os.path.join(PROFILES, "kernel_counts.json")
# the sources that decide what the integrator kernels execute
KERNEL_SOURCES = ["kernels.cuh", "force.cuh", "ferrers.cuh", "dehnen.cuh", "rk32.cuh", "ferrers_table.h"]
OPS = ["dfma", "dmul", "dadd", "ffma", "fmul", "fadd"]
METRICS = [
    "gpu__time_duration.sum", "launch__registers_per_thread", "launch__block_size", "launch__grid_size",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed", "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "dram__bytes_read.sum", "dram__bytes_write.sum",
    "dram__bytes_write.sum.per_second", "sm__cycles_elapsed.avg", "smsp__cycles_active.avg",
    "smsp__average_warp_latency_per_inst_issued.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_dispatch_stall_per_issue_active.ratio",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "smsp__inst_executed_op_shared_atom.sum",
] + ["smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % o for o in OPS]
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def csrc_sha16():
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(HERE, "csrc", f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def raw_page(report):
    """report: an .ncu-rep, or the text `ncu -i REPORT --page raw --csv` wrote (reports are ~20 MB each; gpurun brings back 64 MB)."""
    if report.endswith(".csv"):
        out = open(report).read()
    else:
        out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    head = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    return rows[head], rows[head + 1], rows[head + 2:]


def load_counts():
    if not os.path.exists(COUNTS):
        return {}
    with open(COUNTS) as fh:
        return json.load(fh)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--name", required=True, help="profiles/<name>_ncu_full_summary.csv")
    ap.add_argument("--md", default="", help="the full command that made the report (written to profiles/<name>.md if that file does not exist)")
    ap.add_argument("--counts", default=None, help='key in kernel_counts.json, e.g. "integrate_kernel/barred/f64"')
    ap.add_argument("--work", type=float, default=0.0, help="orbit-steps (or step attempts) integrated by the first profiled launch")
    ap.add_argument("--kernel", default="integrate_kernel", help="substring of the kernel name whose counts are stored")
    a = ap.parse_args()
    names, units, launches = raw_page(a.report)
    col = {n: i for i, n in enumerate(names)}
    kn = col["Kernel Name"]
    os.makedirs(PROFILES, exist_ok=True)
    path = os.path.join(PROFILES, a.name + "_ncu_full_summary.csv")
    with open(path, "w", newline="") as fh:
        w = csv.writer(fh)
        w.writerow(["metric", "unit"] + [r[kn][:60] for r in launches])
        for m in ["Kernel Name", "Block Size", "Grid Size"] + METRICS:
            if m in col:
                w.writerow([m, units[col[m]]] + [r[col[m]] for r in launches])
    print("wrote", path)
    md = os.path.join(PROFILES, a.name + ".md")
    if a.md and not os.path.exists(md):
        with open(md, "w") as fh:
            fh.write("# %s\n\nCommand (under gpurun, after the same command had exited 0 without ncu):\n\n    %s\n\nSummary: `%s`\n"
                     % (a.name, a.md, os.path.basename(path)))
    if a.counts:
        if not a.work > 0:
            raise SystemExit("--counts needs --work (orbit-steps of the profiled launch)")
        r = next(x for x in launches if a.kernel in x[kn])
        cyc = float(r[col["sm__cycles_elapsed.avg"]].replace(",", ""))
        ops = {o: float(r[col["smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % o]].replace(",", "")) * cyc / a.work for o in OPS}
        dram = sum(float(r[col[m]].replace(",", "")) * UNIT_SCALE[units[col[m]]] for m in ("dram__bytes_read.sum", "dram__bytes_write.sum"))
        c = load_counts()
        c[a.counts] = {"per_orbit_step": ops, "dram_bytes_per_launch": dram, "orbit_steps_per_launch": a.work,
                       "kernel": r[kn], "registers": int(r[col["launch__registers_per_thread"]]), "block": r[col["Block Size"]],
                       "duration_ms_under_ncu": float(r[col["gpu__time_duration.sum"]]) * {"ms": 1.0, "us": 1e-3, "s": 1e3, "ns": 1e-6}.get(units[col["gpu__time_duration.sum"]], 1.0),
                       "source": os.path.basename(path), "csrc_sha16": csrc_sha16()}
        with open(COUNTS, "w") as fh:
            json.dump(c, fh, indent=1, sort_keys=True)
        print("updated", COUNTS, a.counts, ops)


if __name__ == "__main__":
    main()
