"""RA-MPPI benchmark: noisy state-steps/s (K*M*T per second) and iterations/s on one B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl reference]

A "step" is one full controller iteration (ra_mppi_step: sample -> nominal + noisy rollouts ->
CVaR -> weights -> update) on the named BASELINE.json workload; default C3 = configs[3]
(K=16384, M=128, T=50, costmap), the configuration BASELINE.json's target is quoted on.
Prints ONE JSON line.  --impl reference times the fp64 oracle.
north_star fixes one GPU, so --gpus N runs N independent replicas (weak scaling); --sharded splits the K samples of
ONE controller over the N ranks instead (strong scaling, one all-gather of 2+2T doubles per rank per step).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2209_12842_b200 import workloads as W  # noqa: E402

METRIC = "noisy_state_steps_per_s"
UNIT = "state-steps/s"

# Algorithmic lane-operations per noisy state-step ("What bounds it"): the instructions the method
# itself needs in its leanest known formulation, one per FP32-lane issue slot (FFMA = 1).
#   Philox4x32-10 call 40 (20 mul-wide + 20 xor3), and a state-step takes n_x/8 of a call (16 bits per uniform, one word per
#   Box-Muller pair): 20 for n_x = 4, 30 for n_x = 6; Box-Muller pair 10 (2 uniforms at 2 each, lg2, sqrt, sin, cos, 2 products);
#   noise add 1 FMA per component; bicycle step 7 (sin, cos, 5 FMA-class); single-track step 75; bilinear lookup 18; racing
#   smooth cost 30.  NOT credited: range reductions, address arithmetic, loop control, the CVaR select, and every circle
#   test (far obstacles are culled exactly, and a culled test is not achieved work).
_BICYCLE = 20 + 20 + 4 + 7
_SINGLE_TRACK = 30 + 30 + 6 + 75
ALGO_OPS = {"PAPER": _BICYCLE + 30, "PAPER-ST": _SINGLE_TRACK + 30, "C0": _BICYCLE, "C1": _BICYCLE, "C2": _SINGLE_TRACK,
            "C3": _BICYCLE + 18, "C4": _BICYCLE}
ALU_PEAK_LANE_OPS = 148 * 128 * 1.965e9  # 148 SMs x 128 FP32 lanes x 1.965 GHz (B200_PROFILING.md nominal)
ISSUE_PEAK_WARP_INST = 148 * 4 * 1.965e9  # one warp instruction per cycle per SM sub-partition
COUNTERS_CSV = os.path.join(ROOT, "profiles", "r3_rollout_counters.csv")
# the sources that decide what noisy_rollout_kernel compiles to; their hash is stored with every capture
ROLLOUT_SOURCES = ("rollout.cuh", "models.cuh", "rng.cuh", "ra_params.cuh", "launchers.h", "rollout_inst.cu")


def rollout_source_sha() -> str:
    """sha256 over the rollout kernel's sources as they are in the tree now (tests/helpers/ncu_counters.py stores the same
    hash in every row it writes, so a capture of an older kernel is recognised and not reported as current)."""
    import hashlib
    h = hashlib.sha256()
    for f in ROLLOUT_SOURCES:
        with open(os.path.join(ROOT, "paper_2209_12842_b200", "csrc", f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read() + b"\0")
    return h.hexdigest()


def kernel_template_args(kernel_name: str):
    """'void noisy_rollout_kernel<0, 1, 0, 2, 0>(...)' -> (0, 1, 0, 2, 0): dynamics, risk, noise variant, slots per lane, half."""
    import re
    m = re.search(r"noisy_rollout_kernel<([^>]*)>", kernel_name or "")
    if not m:
        return None
    conv = lambda t: {"true": 1, "false": 0}.get(t.strip(), None) if t.strip() in ("true", "false") else int(t.strip().split(")")[-1])
    try:
        return tuple(conv(t) for t in m.group(1).split(","))
    except ValueError:
        return None


def capture_status(row, variant=None, scaled=False):
    """Is the committed capture `row` a description of the kernel that is running?  None when there is no row; otherwise
    {"stale": bool, "why": [...], "extrapolated": bool}: stale when the rollout sources have changed since the capture, or
    when the captured instantiation is not the one the live context launches (`variant` = ra_mppi_rollout_variant)."""
    if not row:
        return None
    why = []
    if row.get("source_sha") != rollout_source_sha():
        why.append("rollout kernel sources changed since the capture (source_sha)")
    if variant is not None and kernel_template_args(row.get("kernel", "")) != tuple(variant):
        why.append(f"captured {row.get('kernel', '?')} but the context launches noisy_rollout_kernel<{', '.join(map(str, variant))}>")
    return {"stale": bool(why), "why": why, "extrapolated": bool(scaled)}


def load_counters():
    """Per-launch counters of noisy_rollout_kernel from the committed `ncu --set full` captures (profiles/r3_rollout_counters.md
    names the commands): {workload: {metric: value}}.  Absent file => {} and the derived fractions are null."""
    import csv
    out = {}
    try:
        rows = list(csv.reader(open(COUNTERS_CSV)))
    except OSError:
        return out
    hdr = rows[0]
    for r in rows[1:]:
        if len(r) != len(hdr) or not r[0] or r[0] == "workload":
            continue
        d = {}
        for k, v in zip(hdr[1:], r[1:]):
            if k in ("kernel", "source_sha"):
                d[k] = v
                continue
            try:
                d[k] = float(v.replace(",", ""))
            except ValueError:
                d[k] = v
        out[r[0]] = d
    return out


def counter_key(name: str) -> str:
    """Which capture describes workload `name`: the C4 sweep points share a kernel per M (captured at K = 16384), except
    M = 16 from K = 32768, where a warp carries four samples instead of two (captured at K = 65536)."""
    name = name.upper()
    if name.startswith("C4"):
        parts = name.split("-")
        K = int(parts[1][1:]) if len(parts) > 1 else 8192
        M = parts[2] if len(parts) > 2 else "M64"
        return f"C4-{M}-4PERWARP" if (M == "M16" and K >= 32768) else f"C4-{M}"
    return name


def derived_fractions(name, state_steps, kernel_ms, ffma_peak_tlaneops, counters, variant=None):
    """Roofline fractions of one rollout-kernel launch lasting kernel_ms (measured live):
    frac = algorithmic lane-ops / measured FFMA issue rate (the contract's figure);
    frac_fp32_flop = FP32 flop/s (2 FFMA + FADD + FMUL thread instructions of the ncu capture) / measured FFMA flop/s;
    frac_issue = executed warp instructions (ncu) / issue slots."""
    ops = ALGO_OPS[workload_key(name)] * state_steps
    peak = ffma_peak_tlaneops * 1e12 if ffma_peak_tlaneops and ffma_peak_tlaneops > 0 else ALU_PEAK_LANE_OPS
    out = {"frac": ops / (kernel_ms * 1e-3) / peak, "frac_fp32_flop": None, "frac_issue": None}
    c = counters.get(counter_key(name))
    st = capture_status(c, variant, scaled=bool(c) and c.get("state_steps") != state_steps)
    out["capture"] = st
    if c and not st["stale"]:
        scale = state_steps / c["state_steps"] if c.get("state_steps") else 1.0   # same kernel, different K
        flop = 2.0 * c["smsp__sass_thread_inst_executed_op_ffma_pred_on.sum"] + \
            c["smsp__sass_thread_inst_executed_op_fadd_pred_on.sum"] + c["smsp__sass_thread_inst_executed_op_fmul_pred_on.sum"]
        out["frac_fp32_flop"] = flop * scale / (kernel_ms * 1e-3) / (2.0 * peak)
        out["frac_issue"] = c["smsp__inst_executed.sum"] * scale / (kernel_ms * 1e-3) / ISSUE_PEAK_WARP_INST
    return out


def make_problem(name: str, rank: int = 0) -> W.Problem:
    name = name.upper()
    if name == "C0":
        p = W.config0(near_obstacle=True)
    elif name == "C1":
        p = W.config1()
    elif name == "C2":
        p = W.config2()
    elif name == "C3":
        p = W.config3()
    elif name in ("PAPER", "PAPER-ST"):
        p = W.paper_racing(single_track=name.endswith("ST"))      # the paper's own workload: 3.072e5 trajectories
    elif name.startswith("C4"):
        parts = name.split("-")
        K = int(parts[1][1:]) if len(parts) > 1 else 8192
        M = int(parts[2][1:]) if len(parts) > 2 else 64
        p = W.config4(K=K, M=M)
    else:
        raise SystemExit(f"unknown workload {name}")
    scale = (0.1, 0.5) if p.dyn == W.DYN_BICYCLE else (0.1, 2.0)
    return p.replace(v=W.random_mean_control(p, rank, scale), seed=p.seed + 1000 * rank)


def workload_key(name: str) -> str:
    return name.upper().split("-")[0]


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                     "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80}
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for n, bit in names.items():
                    if r & bit:
                        self.reasons.add(n)
                time.sleep(0.005)
        except Exception as e:  # pragma: no cover
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def cpu_baseline(p: W.Problem, seconds_target: float = 12.0, threads=None):
    """The oracle as it stands, timed on the host cores on a bounded slice of the same workload (threads = None: all
    host cores; 1: the oracle as defined, single-threaded)."""
    from oracle import oracle as O
    orc = O.Oracle(p)
    cores = threads or (os.cpu_count() or 1)
    per_step = 0.13e-6  # rough single-thread cost per state-step; only sizes the sample (CPU-seconds of work)
    n_k = int(min(p.K, max(cores, seconds_target * cores / (per_step * p.M * p.T))))
    t0 = time.perf_counter()
    orc.rollout_costs(k_begin=0, k_end=n_k, n_threads=cores, want_L=False, want_xT=False)
    dt = time.perf_counter() - t0
    return {"value": n_k * p.M * p.T / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"samples k in [0,{n_k}) of {p.name} (K={p.K}, M={p.M}, T={p.T}): {n_k * p.M * p.T} "
                      f"state-steps of O1 (sampling, nominal + noisy rollouts, CVaR) in {dt:.2f} s wall",
            "seconds": dt}


def max_over_ranks(values, world, device):
    """Element-wise MAX of per-rank timings over the process group (a no-op for one rank)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def aggregate_rate(units_per_step, steps, world, max_ms):
    """Whole-job throughput of `world` replicas: all units processed / slowest rank's time."""
    return world * units_per_step * steps / (max_ms * 1e-3)


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step is a bounded slice of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    p = make_problem(args.workload)
    orc = O.Oracle(p)
    cores = os.cpu_count() or 1
    n_k = min(p.K, 64 * cores)
    units = n_k * p.M * p.T
    for _ in range(args.warmup):
        orc.rollout_costs(k_begin=0, k_end=n_k, n_threads=cores, want_L=False, want_xT=False)
    t0 = time.perf_counter()
    for i in range(args.steps):
        orc.rollout_costs(iteration=i, k_begin=0, k_end=n_k, n_threads=cores, want_L=False, want_xT=False)
    dt = time.perf_counter() - t0
    value = units * args.steps / dt
    sample = (f"each step = samples k in [0,{n_k}) of {p.name} ({units} state-steps of O1) on {cores} threads; "
              f"the O2-O3 update needs all K samples and is not in the slice")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{p.name} K={p.K} M={p.M} T={p.T}", "slice": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_cuda(args):
    import torch
    import torch.distributed as dist

    from paper_2209_12842_b200.controller import RaMppi

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2209_12842_b200 import binding as B
    pipe_peaks = B.ra_mppi_measure_pipe_peaks(local)   # measured FFMA / IMAD.WIDE+LOP3 / LOP3 / MUFU rates

    p = make_problem(args.workload, rank)
    if args.materialised:   # the HBM-bound variant: the noise tensor written by the generator, streamed by the rollout kernel
        p = p.replace(noise_mode=W.NOISE_MATERIALISED)
    ctl = RaMppi(p, device=local)
    dev = ctl.device
    d_x0 = ctl.tensor(p.x0)
    v_init = ctl.tensor(p.v)
    d_v = v_init.clone()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        d_v.copy_(v_init)
        ctl.step(d_x0, d_v, i)
    barrier()

    # ---- device-resident timing: one event pair per step on the launching stream, L2 flushed between
    sampler = ClockSampler(local)
    sampler.start()
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    stops = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    barrier()
    t_wall0 = time.perf_counter()
    for i in range(args.steps):
        d_v.copy_(v_init)
        flush.zero_()
        starts[i].record(stream)
        ctl.step(d_x0, d_v, args.warmup + i)
        stops[i].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    sampler.stop_flag = True
    sampler.join()
    ms = np.array([s.elapsed_time(e) for s, e in zip(starts, stops)])
    total_ms = float(ms.sum())

    # ---- roofline pass: event pair around the fused rollout kernel itself
    ctl.enable_kernel_timing(True)
    kms = []
    for i in range(min(args.steps, 50)):
        d_v.copy_(v_init)
        flush.zero_()
        ctl.step(d_x0, d_v, args.warmup + i)
        kms.append(ctl.last_rollout_ms())
    ctl.enable_kernel_timing(False)
    kernel_ms = float(np.mean(kms))

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D x0,v -> step -> D2H v+
    h_x0 = torch.tensor(np.asarray(p.x0, dtype=np.float32)).pin_memory()
    h_v0 = torch.tensor(np.asarray(p.v, dtype=np.float32)).pin_memory()
    h_v = h_v0.clone().pin_memory()
    for i in range(3):
        h_v.copy_(h_v0)
        ctl.step_host(h_x0, h_v, i)
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        h_v.copy_(h_v0)
        ctl.step_host(h_x0, h_v, args.warmup + i)   # returns after the D2H copy of v+ has landed
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0

    # ---- max over ranks; every rank is an independent replica of the same workload (weak scaling)
    total_ms, e2e_ms, kernel_ms = max_over_ranks([total_ms, e2e_s * 1e3, kernel_ms], world, dev)
    units_step = p.state_steps
    value = aggregate_rate(units_step, args.steps, world, total_ms)
    e2e_value = aggregate_rate(units_step, args.steps, world, e2e_ms)

    if rank == 0:
        key = workload_key(args.workload)
        counters = load_counters()
        ops = ALGO_OPS[key] * units_step
        achieved = ops / (kernel_ms * 1e-3)
        peak = pipe_peaks["ffma"] * 1e12 if pipe_peaks.get("ffma", 0) > 0 else ALU_PEAK_LANE_OPS
        fr = derived_fractions(args.workload, units_step, kernel_ms, pipe_peaks.get("ffma"), counters, ctl.rollout_variant)
        stale = bool(fr["capture"] and fr["capture"]["stale"])
        c = {} if stale else counters.get(counter_key(args.workload), {})   # a stale capture describes another kernel: report nothing from it
        pct = lambda k: (c[k] / 100.0 if k in c else None)
        traffic = (c["dram__bytes_read.sum"] + c["dram__bytes_write.sum"]) if "dram__bytes_read.sum" in c else None
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{p.name} K={p.K} M={p.M} T={p.T}", "baseline_config_index": int(key[1]) if key[1:].isdigit() else None,
                       "l2_flush_between_steps": True, "parallelism": "replicas only" if world > 1 else "single GPU",
                       "noise_mode": "materialised" if args.materialised else "fused"},
            "iterations_per_s": world * args.steps / (total_ms * 1e-3),
            "wall_ms_per_step_incl_flush": 1e3 * t_wall / args.steps,
            "clocks": sampler.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(4 * (8 + 2 * p.T)),
                    "d2h_bytes_per_step": int(4 * 2 * p.T), "ms_per_step": e2e_ms / args.steps,
                    "api": "ra_mppi_step_host (pinned host x0, v -> v+)"},
            "gpu_launches": int(ctl.launches_per_step * args.steps),
            "roofline": {
                "bound": "issue+xu", "kernel": "noisy_rollout_kernel",
                "bound_note": "plain SM pipes, no tensor or HBM bound: instruction issue slots and the XU (MUFU) pipe co-limit (the contract's 'alu' class)",
                "binding_resource": "issue slots and the XU (MUFU) pipe, co-limiting; fmaheavy behind them (pipe_busy)",
                "achieved": achieved / 1e12, "peak": peak / 1e12,
                "unit": "Tlane-op/s (algorithmic instructions per FP32-lane issue slot; FFMA = 1)",
                "frac": achieved / peak,
                "frac_definition": "useful-instruction issue slots: the method's algorithmic instructions (Philox integer work, MUFU and FP32 "
                                   "each counted as one FP32-lane slot) per second / measured FFMA issue rate.  NOT the literal FP32 figure: "
                                   "that is frac_fp32_flop (FP32 flop/s / FP32 peak); frac_issue counts every executed instruction",
                # the same launch on the stricter readings: FP32 flop only, and all executed instructions
                "frac_fp32_flop": fr["frac_fp32_flop"],
                "fp32_flop_note": "(2 FFMA + FADD + FMUL thread instructions per launch, ncu SASS counters of the committed capture) / "
                                  "live kernel time / (2 x measured FFMA rate); Philox integer work and MUFU are not FP32 flop",
                "frac_issue": fr["frac_issue"],
                "pipe_busy": {"issue": pct("smsp__issue_active.avg.pct_of_peak_sustained_active"),
                              "fmaheavy": pct("sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed"),
                              "fma": pct("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active"),
                              "alu": pct("sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active"),
                              "xu": pct("sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active"),
                              "source": "ncu --set full capture, profiles/r3_rollout_counters.csv" if c else None},
                "traffic": traffic,
                # frac_fp32_flop, frac_issue, pipe_busy and traffic come from a committed ncu capture scaled by the live kernel time;
                # they are null, and this is true, when the rollout sources or the launched instantiation differ from the captured ones
                "stale_capture": stale, "capture": fr["capture"],
                "nominal_peak": ALU_PEAK_LANE_OPS / 1e12, "frac_of_nominal": achieved / ALU_PEAK_LANE_OPS,
                "measured_pipe_peaks_Tlaneops": pipe_peaks,
                "algorithmic_ops_per_state_step": ALGO_OPS[key], "kernel_ms": kernel_ms,
                "kernel_share_of_step": kernel_ms / (total_ms / args.steps),
                "peak_source": "measured in this run: FFMA issue rate of ra_mppi_measure_pipe_peaks (FFMA = 1 lane-op); "
                               "nominal = 148 SMs x 128 FP32 lanes x 1.965 GHz (DESIGN.md)"},
        }
        if world == 1 and not args.no_workloads:
            line["workloads"] = run_workloads(pipe_peaks.get("ffma"), counters, flush, with_cpu=not args.no_cpu_baseline)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(p)
            line["cpu_baseline_1thread"] = cpu_baseline(p, seconds_target=6.0, threads=1)
        print(json.dumps(line))
    ctl.close()
    if world > 1:
        dist.destroy_process_group()


def run_sharded(args):
    """--sharded: ONE controller whose K samples are split over the N ranks (strong scaling).
    Every step = local rollouts + partial reduction, one NCCL all-gather of 2+2T doubles per rank, combine."""
    import torch
    import torch.distributed as dist

    from paper_2209_12842_b200.sharded import ShardedRaMppi

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    p = make_problem(args.workload, 0)              # the same problem on every rank; each takes its K-shard
    sc = ShardedRaMppi(p, device=local)
    dev = sc.ctl.device
    d_x0, v_init = sc.ctl.tensor(p.x0), sc.ctl.tensor(p.v)
    d_v = v_init.clone()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        d_v.copy_(v_init)
        sc.step(d_x0, d_v, i)
    sampler = ClockSampler(local)
    sampler.start()
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    stops = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    barrier()
    for i in range(args.steps):
        d_v.copy_(v_init)
        flush.zero_()
        starts[i].record(stream)
        sc.step(d_x0, d_v, args.warmup + i)
        stops[i].record(stream)
    barrier()
    sampler.stop_flag = True
    sampler.join()
    total_ms = float(sum(s.elapsed_time(e) for s, e in zip(starts, stops)))
    # end to end: pinned host x0, v -> device, sharded step, v+ -> host, every step
    h_x0 = torch.tensor(np.asarray(p.x0, dtype=np.float32)).pin_memory()
    h_v0 = torch.tensor(np.asarray(p.v, dtype=np.float32)).pin_memory()
    h_v = h_v0.clone().pin_memory()
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        d_x0.copy_(h_x0, non_blocking=True)
        d_v.copy_(h_v0, non_blocking=True)
        sc.step(d_x0, d_v, args.warmup + i)
        h_v.copy_(d_v, non_blocking=True)
        torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    total_ms, e2e_ms = max_over_ranks([total_ms, e2e_ms], world, dev)
    if rank == 0:
        units = p.state_steps                       # the whole problem, once: strong scaling
        print(json.dumps({
            "metric": METRIC, "value": units * args.steps / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{p.name} K={p.K} M={p.M} T={p.T}", "l2_flush_between_steps": True,
                       "parallelism": f"K-sharded over {world} GPU(s): {sc.ctl.K} samples on rank 0, "
                                      f"one all-gather of {8 * (2 + 2 * p.T)} B per rank per step"},
            "iterations_per_s": args.steps / (total_ms * 1e-3), "clocks": sampler.summary(),
            "e2e": {"value": units * args.steps / (e2e_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(4 * (p.nx + 2 * p.T)), "d2h_bytes_per_step": int(4 * 2 * p.T),
                    "ms_per_step": e2e_ms / args.steps, "api": "ShardedRaMppi.step (pinned host x0, v -> v+)"},
            "gpu_launches": int((sc.ctl.launches_per_step + 1) * args.steps),
        }))
    sc.close()
    if world > 1:
        dist.destroy_process_group()


def quick_time(p, steps=50, warmup=5, flush=None):
    """Device-timed ra_mppi_step on problem p (events per step, L2 flushed between); helper of the `workloads` array."""
    import torch

    from paper_2209_12842_b200.controller import RaMppi
    ctl = RaMppi(p, device=0)
    d_x0, v_init = ctl.tensor(p.x0), ctl.tensor(p.v)
    d_v = v_init.clone()
    if flush is None:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=ctl.device)
    stream = torch.cuda.current_stream()
    ms, kms = [], []
    for timed in (False, True):     # a plain pass for the step time, then one with the event pair around the rollout kernel
        ctl.enable_kernel_timing(timed)
        for i in range(warmup + steps):
            d_v.copy_(v_init)
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctl.step(d_x0, d_v, i)
            b.record(stream)
            b.synchronize()
            if i >= warmup:
                (kms if timed else ms).append(ctl.last_rollout_ms() if timed else a.elapsed_time(b))
    variant = list(ctl.rollout_variant)
    ctl.close()
    step_ms = float(np.mean(ms))
    return {"workload": f"{p.name} K={p.K} M={p.M} T={p.T}", "ms_per_step": step_ms, "iterations_per_s": 1e3 / step_ms,
            "state_steps_per_s": p.state_steps / (step_ms * 1e-3), "rollout_kernel_ms": float(np.mean(kms)),
            "rollout_variant": variant}


def run_workloads(ffma_peak, counters, flush=None, with_cpu=False):
    """Every workload BASELINE.json names, on this GPU, each with its roofline fractions (north_star: "throughput on the
    five synthetic workloads ... as a fraction of the relevant roofline"): configs 0-3, the 12 points of the config-4
    sweep, the paper's own workload (two vehicle models), the materialised-noise (HBM-bound) variant of C3, and the
    500-iteration CUDA-graph closed loop of config 4."""
    import torch

    from paper_2209_12842_b200.controller import RaMppi
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    out = []

    def add(tag, name, p=None, steps=30):
        p = make_problem(name) if p is None else p
        r = quick_time(p, steps=steps, flush=flush)
        r.update({"kind": tag, "name": name})
        r.update(derived_fractions(name, p.state_steps, r["rollout_kernel_ms"], ffma_peak, counters, r["rollout_variant"]))
        r["roofline_bound"] = "issue+xu"
        out.append(r)
        return r, p

    for name in ("C0", "C1", "C2", "C3"):
        r, p = add("BASELINE config", name)
        if with_cpu:   # the oracle as defined (one thread) on a ~1 s slice of this config, beside the GPU number
            r["cpu_oracle_1thread"] = cpu_baseline(p, seconds_target=1.0, threads=1)
    for name in ("PAPER", "PAPER-ST"):   # the paper's own workload (context for its 44.3 Hz on an RTX 3090)
        add("paper workload (1024 x 300 x 30, costs (20)-(23), l = q)", name, steps=50)
    for K in W.C4_SWEEP_K:
        for M in W.C4_SWEEP_M:
            add("config 4 sweep", f"C4-K{K}-M{M}", steps=15 if K * M >= 65536 * 64 else 30)
    # materialised-noise mode: w[K,T,n_x,M] written by the generator and streamed back by the rollout kernel
    p = make_problem("C3").replace(noise_mode=W.NOISE_MATERIALISED)
    r = quick_time(p, steps=15, flush=flush)
    noise_bytes = 4.0 * p.nx * p.state_steps
    gbs = noise_bytes / (r["rollout_kernel_ms"] * 1e-3) / 1e9
    r.update({"kind": "materialised noise (HBM-bound variant of C3)", "name": "C3-materialised", "roofline_bound": "hbm",
              "noise_tensor_GB": noise_bytes / 1e9, "rollout_read_GBps": gbs, "hbm_peak_GBps": hbm_peak,
              "peak_source": "measured (MEASURED_PEAKS.json)" if peaks else "fallback", "frac": gbs / hbm_peak,
              "frac_note": "rollout kernel streaming the noise tensor: algorithmic bytes 4 n_x K M T / kernel time / HBM copy peak"})
    # the write side: the generator fills the same tensor once per step.  Its time is the step minus the rollout kernel, which
    # also contains the sampling, nominal-rollout and update kernels (about 0.03 ms here), so the rate is a lower bound
    gen_ms = r["ms_per_step"] - r["rollout_kernel_ms"]
    # a write-only stream does not reach the copy peak (which counts bytes read + bytes written): the ceiling of a kernel that
    # only writes is measured here with a plain device fill of a buffer larger than L2
    fill = flush if flush is not None else torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    for _ in range(3):
        fill.zero_()
    ev[0].record()
    for _ in range(10):
        fill.zero_()
    ev[1].record()
    ev[1].synchronize()
    write_peak = fill.numel() * 10 / (ev[0].elapsed_time(ev[1]) * 1e-3) / 1e9
    r.update({"generator_ms_upper_bound": gen_ms, "generator_write_GBps": noise_bytes / (gen_ms * 1e-3) / 1e9,
              "generator_frac": noise_bytes / (gen_ms * 1e-3) / 1e9 / hbm_peak,
              "hbm_write_only_GBps": write_peak, "generator_frac_of_write_only": noise_bytes / (gen_ms * 1e-3) / 1e9 / write_peak,
              "generator_note": "materialise_noise_kernel writes the tensor once per step: bytes / (step - rollout kernel) / HBM copy peak; "
                                "a lower bound (the difference also holds the three small kernels).  hbm_write_only_GBps = a device fill of 256 MB timed in this run: "
                                "the ceiling of a write-only stream, about 0.6 of the copy peak"})
    out.append(r)
    # closed loop: config 4, K=8192, M=64, 500 receding-horizon iterations replayed from one CUDA graph
    name = "C4-K8192-M64"
    p = make_problem(name)
    ctl = RaMppi(p, device=0)
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    ctl.closed_loop(d_x0, d_v, 0, 20)                      # capture + warm-up
    d_x0.copy_(ctl.tensor(p.x0)); d_v.zero_()
    log, ms = ctl.closed_loop(d_x0, d_v, 0, 500)           # per-iteration events: p50/p99
    d_x0.copy_(ctl.tensor(p.x0)); d_v.zero_()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(torch.cuda.current_stream())
    ctl.closed_loop(d_x0, d_v, 0, 500, log=False, timing=False)   # sustained: no per-iteration events
    b.record(torch.cuda.current_stream())
    b.synchronize()
    total = a.elapsed_time(b)
    log = log.cpu().numpy()
    p50 = float(np.percentile(ms, 50))
    cl = {"kind": "closed loop (one CUDA graph launch per iteration)", "name": name + "-closed-loop",
          "workload": f"{p.name} K={p.K} M={p.M} T={p.T}", "iterations": 500, "sustained_hz": 500.0 / (total * 1e-3),
          "latency_ms_p50": p50, "latency_ms_p99": float(np.percentile(ms, 99)), "latency_ms_max": float(ms.max()),
          "ms_per_step": total / 500.0, "state_steps_per_s": p.state_steps * 500.0 / (total * 1e-3),
          "final_state": [float(x) for x in log[-1, :p.nx]],
          "distance_travelled_m": float(np.hypot(np.diff(log[:, 0]), np.diff(log[:, 1])).sum()), "roofline_bound": "issue+xu"}
    # whole-iteration fractions (the graph has no event pair around the rollout kernel): iteration time as the denominator
    cl.update(derived_fractions(name, p.state_steps, total / 500.0, ffma_peak, counters, ctl.rollout_variant))
    cl["frac_note"] = "whole iteration (sampling + rollouts + update + plant) as the time base"
    out.append(cl)
    ctl.close()
    return out


def run_report(args):
    """--report: the `workloads` array of the default line, one JSON object per line (not the driver's bench line)."""
    from paper_2209_12842_b200 import binding as B
    pipe_peaks = B.ra_mppi_measure_pipe_peaks(0)
    for r in run_workloads(pipe_peaks.get("ffma"), load_counters()):
        print(json.dumps({"report": r.pop("kind"), **r}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--report", action="store_true", help="all workloads + sweep + closed loop (not the bench line)")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-workloads", action="store_true", help="leave the per-workload array out of the line (short profiling runs)")
    ap.add_argument("--materialised", action="store_true",
                    help="time the materialised-noise (HBM-bound) variant of the workload instead of the fused one")
    ap.add_argument("--sharded", action="store_true",
                    help="one controller, K split over the ranks (strong scaling) instead of N independent replicas")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    if args.report:
        run_report(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.sharded:
        run_sharded(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
