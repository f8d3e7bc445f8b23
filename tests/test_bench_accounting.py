"""Host-side checks of bench.py's roofline accounting (no GPU): every workload of the `workloads` array finds its row in the
committed ncu counter table, and the three fractions are what their definitions say."""
import os

import pytest

import bench
from paper_2209_12842_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_every_workload_has_a_counter_row():
    counters = bench.load_counters()
    assert counters, "profiles/r3_rollout_counters.csv is missing or empty"
    names = ["C0", "C1", "C2", "C3", "PAPER", "PAPER-ST", "C4-K8192-M64"] + \
        [f"C4-K{K}-M{M}" for K in W.C4_SWEEP_K for M in W.C4_SWEEP_M]
    for n in names:
        key = bench.counter_key(n)
        assert key in counters, (n, key)
        c = counters[key]
        for m in ("state_steps", "smsp__inst_executed.sum", "smsp__sass_thread_inst_executed_op_ffma_pred_on.sum",
                  "smsp__sass_thread_inst_executed_op_fadd_pred_on.sum", "smsp__sass_thread_inst_executed_op_fmul_pred_on.sum",
                  "dram__bytes_read.sum", "smsp__issue_active.avg.pct_of_peak_sustained_active"):
            assert isinstance(c[m], float) and c[m] >= 0, (n, m, c.get(m))
    # the M = 16 kernel differs by K (four samples per warp from K = 32768): two rows, not one
    assert bench.counter_key("C4-K65536-M16") != bench.counter_key("C4-K16384-M16") == bench.counter_key("C4-K1024-M16")
    assert bench.counter_key("C4-K65536-M256") == bench.counter_key("C4-K1024-M256")


def test_fractions_follow_their_definitions():
    counters = bench.load_counters()
    p = bench.make_problem("C3")
    c = counters["C3"]
    assert c["state_steps"] == p.state_steps == 16384 * 128 * 50
    kernel_ms, ffma_peak = 0.35, 35.4            # Tlane-op/s
    f = bench.derived_fractions("C3", p.state_steps, kernel_ms, ffma_peak, counters)
    assert f["frac"] == pytest.approx(bench.ALGO_OPS["C3"] * p.state_steps / 0.35e-3 / 35.4e12)
    flop = 2 * c["smsp__sass_thread_inst_executed_op_ffma_pred_on.sum"] + c["smsp__sass_thread_inst_executed_op_fadd_pred_on.sum"] + \
        c["smsp__sass_thread_inst_executed_op_fmul_pred_on.sum"]
    assert f["frac_fp32_flop"] == pytest.approx(flop / 0.35e-3 / (2 * 35.4e12))
    assert f["frac_issue"] == pytest.approx(c["smsp__inst_executed.sum"] / 0.35e-3 / (148 * 4 * 1.965e9))
    assert 0 < f["frac_fp32_flop"] < f["frac"] < 1 and 0 < f["frac_issue"] < 1
    # a sweep point scales its capture's counts by K
    f1 = bench.derived_fractions("C4-K4096-M64", 4096 * 64 * 50, 0.08, ffma_peak, counters)
    f2 = bench.derived_fractions("C4-K16384-M64", 16384 * 64 * 50, 0.32, ffma_peak, counters)
    assert f1["frac_issue"] == pytest.approx(f2["frac_issue"]) and f1["frac_fp32_flop"] == pytest.approx(f2["frac_fp32_flop"])
    # no capture -> the contract's fraction only
    f3 = bench.derived_fractions("C3", p.state_steps, kernel_ms, ffma_peak, {})
    assert f3["frac"] == f["frac"] and f3["frac_fp32_flop"] is None and f3["frac_issue"] is None


def test_capture_belongs_to_the_sources_in_the_tree(monkeypatch):
    """The ncu-derived fractions are only reported for the kernel they were captured from: every row of the committed table
    carries the hash of the rollout sources it was taken on, which must be the hash of the tree; a changed source, or a
    context that launches another instantiation than the captured one, turns the derived fractions into nulls."""
    counters = bench.load_counters()
    sha = bench.rollout_source_sha()
    for key, row in counters.items():
        assert row["source_sha"] == sha, f"{key}: the capture is of other sources -- re-capture (profiles/r3_rollout_counters.md)"
    p = bench.make_problem("C3")
    assert bench.kernel_template_args(counters["C3"]["kernel"]) == (0, 1, 0, 2, 0)     # bicycle, costmap, Gaussian, 2 slots, whole warp
    ok = bench.derived_fractions("C3", p.state_steps, 0.35, 35.4, counters, variant=(0, 1, 0, 2, 0))
    assert ok["capture"] == {"stale": False, "why": [], "extrapolated": False} and ok["frac_issue"] is not None
    other = bench.derived_fractions("C3", p.state_steps, 0.35, 35.4, counters, variant=(0, 1, 0, 4, 0))
    assert other["capture"]["stale"] and other["frac_issue"] is None and other["frac_fp32_flop"] is None and other["frac"] == ok["frac"]
    scaled = bench.derived_fractions("C4-K4096-M64", 4096 * 64 * 50, 0.08, 35.4, counters)
    assert scaled["capture"]["extrapolated"] and not scaled["capture"]["stale"]
    monkeypatch.setattr(bench, "rollout_source_sha", lambda: "0" * 64)                 # as if rollout.cuh had been edited
    touched = bench.derived_fractions("C3", p.state_steps, 0.35, 35.4, counters, variant=(0, 1, 0, 2, 0))
    assert touched["capture"]["stale"] and "source_sha" in touched["capture"]["why"][0]
    assert touched["frac_issue"] is None and touched["frac_fp32_flop"] is None


def test_algorithmic_op_counts_match_design():
    # half a Philox call 20, two Box-Muller pairs 20, noise add 4, bicycle step 7, bilinear 18
    assert bench.ALGO_OPS["C3"] == 20 + 20 + 4 + 7 + 18 == 69
    assert bench.ALGO_OPS["C1"] == bench.ALGO_OPS["C4"] == bench.ALGO_OPS["C0"] == 51
    assert bench.ALGO_OPS["C2"] == 30 + 30 + 6 + 75 == 141
