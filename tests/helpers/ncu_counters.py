"""Compact per-launch counter table from `ncu --set full` reports of the rollout kernel (roofline accounting of bench.py).

    python tests/helpers/ncu_counters.py WORKLOAD=report.ncu-rep [WORKLOAD=report.ncu-rep ...] > profiles/<name>.csv

Runs `ncu -i <report> --page raw --csv` (no GPU needed) for every report, keeps the first profiled launch and the metrics
below, and prefixes each row with the workload name and its noisy state-steps per launch (K*M*T, from bench.make_problem).
bench.py reads the table for `roofline.frac_fp32_flop`, `frac_issue`, `pipe_busy` and `traffic`; the instruction counts are
per launch, so bench.py divides them by the kernel time it measures live.  Every row carries `source_sha`, the hash of the
rollout kernel's sources at the time the table is written (bench.rollout_source_sha): run this straight after the capture, on
the tree that was profiled.  bench.py nulls the derived fractions when the hash or the kernel instantiation no longer matches.
A development tool, not part of the package; no arithmetic of the method lives here.
"""
from __future__ import annotations

import csv
import io
import os
import subprocess
import sys

METRICS = [
    "gpu__time_duration.sum",
    "launch__registers_per_thread",
    "launch__grid_size",
    "smsp__inst_executed.sum",
    "smsp__sass_thread_inst_executed_op_ffma_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_fadd_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_fmul_pred_on.sum",
    "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active",
    "dram__bytes_read.sum",
    "dram__bytes_write.sum",
    "l1tex__t_sector_hit_rate.pct",
]
_UNIT_SCALE = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0, "msecond": 1e3, "ms": 1e3, "us": 1.0, "usecond": 1.0,
               "ns": 1e-3, "nsecond": 1e-3, "second": 1e6, "s": 1e6}


def read_report(path):
    raw = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr, units, vals = rows[0], rows[1], rows[2]
    col = {h: i for i, h in enumerate(hdr)}
    out = {"kernel": vals[col["Kernel Name"]]}
    for m in METRICS:
        if m not in col:
            out[m] = ""
            continue
        v = float(vals[col[m]].replace(",", "")) if vals[col[m]] not in ("", "no data") else float("nan")
        u = units[col[m]]
        if m.startswith("dram__bytes") or m == "gpu__time_duration.sum":
            v *= _UNIT_SCALE.get(u, 1.0)     # bytes, microseconds
        out[m] = v
    return out


def main(argv):
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
    import bench
    sha = bench.rollout_source_sha()
    w = csv.writer(sys.stdout, lineterminator="\n")
    w.writerow(["workload", "state_steps", "kernel", "source_sha"] + METRICS)
    for arg in argv:
        name, path = arg.split("=", 1)
        r = read_report(path)
        p = bench.make_problem(name)
        w.writerow([bench.counter_key(name), p.state_steps, r["kernel"], sha] + [r[m] for m in METRICS])


if __name__ == "__main__":
    main(sys.argv[1:])
