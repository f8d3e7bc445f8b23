"""Closed-loop glue (A10) and host-buffer entry point, through the C ABI (pytest -m gpu).

The 500-iteration trajectory is not compared as a whole (feedback amplifies rounding):
parity is teacher-forced -- at chosen iterations the GPU's (x0, v, iteration) is handed to the
oracle and that single step is compared.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import workloads as W

from parity_utils import TOL_STATE_ABS, TOL_V_ABS, check_rollout_parity, check_step_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    from paper_2209_12842_b200 import build
    build.build()
    return torch


def _ctl(p):
    from paper_2209_12842_b200.controller import RaMppi
    return RaMppi(p, device=0)


@pytest.mark.parametrize("cfg", ["bicycle", "single_track"])
def test_plant_and_shift(torch_cuda, cfg):
    torch = torch_cuda
    p = W.small(W.config4(), K=64, M=32, T=17) if cfg == "bicycle" else W.small(W.config2(), K=32, M=32, T=9)
    ctl, orc = _ctl(p), O.Oracle(p)
    v = W.random_mean_control(p, 3, (0.3, 4.0))          # includes values beyond the clamps
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(v)
    for it in (0, 7, 499):
        x_before = d_x0.cpu().numpy().astype(np.float64)
        v_before = d_v.cpu().numpy().astype(np.float64)
        u = ctl.plant_shift(d_x0, d_v, it)
        torch.cuda.synchronize()
        assert np.array_equal(u.cpu().numpy(), v_before[0].astype(np.float32))        # applied control = v+_0
        ref_x = orc.plant_step(x_before, v_before[0], it)
        assert np.abs(d_x0.cpu().numpy() - ref_x).max() < 1e-5
        assert np.array_equal(d_v.cpu().numpy(), O.shift(v_before).astype(np.float32))  # warm-start shift, exact


def test_closed_loop_graph_teacher_forced(torch_cuda):
    torch = torch_cuda
    p = W.small(W.config4(), K=512, M=64, T=50)
    ctl, orc = _ctl(p), O.Oracle(p)
    n_iter, it0 = 40, 3
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    log, ms = ctl.closed_loop(d_x0, d_v, it0, n_iter)
    torch.cuda.synchronize()
    log = log.cpu().numpy()
    assert ms.shape == (n_iter,) and (ms > 0).all()
    assert np.isfinite(log).all()
    assert np.array_equal(log[-1, :4], d_x0.cpu().numpy())
    # the graph replay equals the same sequence issued call by call (same kernels, same counters)
    e_x0, e_v = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    checkpoints = {}
    for i in range(n_iter):
        if i in (0, 1, 2, 10, n_iter - 1):
            checkpoints[i] = (e_x0.cpu().numpy().astype(np.float64), e_v.cpu().numpy().astype(np.float64))
        ctl.step(e_x0, e_v, it0 + i)
        u = ctl.plant_shift(e_x0, e_v, it0 + i)
        torch.cuda.synchronize()
        assert np.array_equal(log[i, :4], e_x0.cpu().numpy()), i
        assert np.array_equal(log[i, 4:], u.cpu().numpy()), i
    assert np.array_equal(e_v.cpu().numpy(), d_v.cpu().numpy())
    # teacher-forced single steps against the oracle
    for i, (x0, v) in checkpoints.items():
        g, r = check_rollout_parity(p, ctl, orc, iteration=it0 + i, x0=x0, v=v, k_begin=0, k_end=96)
        rf = orc.rollout_costs(x0=x0, v=v, iteration=it0 + i, n_threads=8, want_L=False, want_xT=False)
        verdict, err = check_step_parity(p, ctl, orc, rf, iteration=it0 + i, x0=x0, v=v)
        print(f"iteration {it0 + i}: v+ {verdict}")
    # the car makes progress along the track and stays near the lane
    assert np.hypot(log[-1, 0] - p.x0[0], log[-1, 1] - p.x0[1]) > 2.0
    # second call re-uses the cached graph and restarts the counter
    d_x0b, d_vb = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    d_x0.copy_(d_x0b); d_v.copy_(d_vb)
    log2, _ = ctl.closed_loop(d_x0, d_v, it0, n_iter)
    torch.cuda.synchronize()
    assert np.array_equal(log2.cpu().numpy(), log)


def test_closed_loop_config4_at_its_stated_size(torch_cuda):
    """BASELINE config 4 as stated and as bench.py times it: K = 8192, M = 64, T = 50, 500 receding-horizon iterations
    replayed from one CUDA graph (Alg.1 l.1-2, 31-33).  At this K the update kernel takes four
    sample ranges and its last CTA combines them and applies the plant and the shift, which the K = 512 case above does
    not reach.  The whole replay must equal the same 500 iterations issued call by call, bit for bit; and at iterations
    {0, 1, 2, 10, 100, 499} the loop's own (x0, v, iteration) is handed to the oracle and that single step compared
    (SURVEY.md section 8(c) item 6): stage-wise on a 96-sample slice, S~ and v+ on all K samples."""
    torch = torch_cuda
    import bench
    p = bench.make_problem("C4-K8192-M64")
    assert (p.K, p.M, p.T) == (8192, 64, 50)
    ctl, orc = _ctl(p), O.Oracle(p)
    n_iter, marks = 500, (0, 1, 2, 10, 100, 499)
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    log, _ = ctl.closed_loop(d_x0, d_v, 0, n_iter, timing=False)
    # call by call, keeping the trajectory on the device; the host looks only at the marked iterations
    e_x0, e_v = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    xs = torch.empty(n_iter, p.nx + 2, device=e_x0.device)
    checkpoints = {}
    for i in range(n_iter):
        if i in marks:
            checkpoints[i] = (e_x0.cpu().numpy().astype(np.float64), e_v.cpu().numpy().astype(np.float64))
        ctl.step(e_x0, e_v, i)
        u = ctl.plant_shift(e_x0, e_v, i)
        xs[i, :p.nx].copy_(e_x0)
        xs[i, p.nx:].copy_(u)
    torch.cuda.synchronize()
    assert torch.isfinite(log).all()
    diff = (log != xs).any(dim=1).nonzero()
    assert diff.numel() == 0, f"graph replay and call-by-call differ first at iteration {int(diff[0])}"
    assert torch.equal(e_v, d_v) and torch.equal(e_x0, d_x0)
    for i, (x0, v) in checkpoints.items():
        g, r = check_rollout_parity(p, ctl, orc, iteration=i, x0=x0, v=v, k_begin=4090, k_end=4186)   # across two ranges
        rf = orc.rollout_costs(x0=x0, v=v, iteration=i, n_threads=O.host_cores(), want_L=False, want_xT=False)
        gs = g["S_tilde"]
        from parity_utils import assert_costs_close
        assert_costs_close(gs, rf["S_tilde"], f"S_tilde over all K at iteration {i}")
        verdict, err = check_step_parity(p, ctl, orc, rf, iteration=i, x0=x0, v=v,
                                         case=f"config-4 closed loop K=8192 M=64 T=50, iteration {i} of 500 (teacher-forced)")
        print(f"iteration {i}: x0 = {np.round(x0, 3)}, risk active on {(rf['cvar'] > 0).mean():.2f} of samples, v+ {verdict}, err {err:.2e}")
    ctl.close()


def test_step_host_equals_step(torch_cuda):
    torch = torch_cuda
    p = W.small(W.config3(), K=256, M=128, T=50)
    p = p.replace(v=W.random_mean_control(p, 1))
    ctl = _ctl(p)
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(p.v)
    ctl.step(d_x0, d_v, 5)
    torch.cuda.synchronize()
    h_x0 = torch.tensor(np.asarray(p.x0, dtype=np.float32)).pin_memory()
    h_v = torch.tensor(np.asarray(p.v, dtype=np.float32)).pin_memory()
    ctl.step_host(h_x0, h_v, 5)
    assert np.array_equal(h_v.numpy(), d_v.cpu().numpy())
    # pageable numpy memory works too
    h_v2 = torch.tensor(np.asarray(p.v, dtype=np.float32))
    ctl.step_host(torch.tensor(np.asarray(p.x0, dtype=np.float32)), h_v2, 5)
    assert np.array_equal(h_v2.numpy(), d_v.cpu().numpy())


def test_kernel_timing_hook(torch_cuda):
    torch = torch_cuda
    p = W.small(W.config3(), K=1024, M=128, T=50)
    ctl = _ctl(p)
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(p.v)
    ctl.enable_kernel_timing(True)
    ctl.step(d_x0, d_v, 0)
    ms = ctl.last_rollout_ms()
    assert 0.0 < ms < 100.0
    assert ctl.launches_per_step == 4   # sampling, nominal rollout, noisy rollouts, weights/update


def test_step_is_capturable_in_a_caller_graph(torch_cuda):
    """include/ra_mppi.h: ra_mppi_step only enqueues (no sync, no allocation), side-stream fork/join included,
    so a caller can capture it in its own CUDA graph; replays reproduce the eager result bit for bit."""
    torch = torch_cuda
    p = W.small(W.config1(), K=300, M=64, T=30)
    p = p.replace(v=W.random_mean_control(p, 1))
    ctl = _ctl(p)
    d_x0, v0 = ctl.tensor(p.x0), ctl.tensor(p.v)
    v_eager = v0.clone()
    ctl.step(d_x0, v_eager, 5)
    torch.cuda.synchronize()
    v_graph = v0.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):                      # captures on torch's side stream; RaMppi uses the current stream
        ctl.step(d_x0, v_graph, 5)
    for _ in range(3):
        v_graph.copy_(v0)
        g.replay()
    torch.cuda.synchronize()
    assert torch.equal(v_graph, v_eager)
    ctl.close()


def test_step_host_graph_follows_set_env_and_timing_mode(torch_cuda):
    """ra_mppi_step_host submits one captured graph per call: the capture must be dropped when the environment changes,
    and the call-by-call path a timed step takes (plain launches, no programmatic dependent launch) must give the same bits."""
    torch = torch_cuda
    p = W.small(W.config1(), K=160, M=64, T=25)
    p = p.replace(v=W.random_mean_control(p, 2))
    moved = p.circles + np.array([0.1, -0.05, 0.02])
    a, b = _ctl(p), _ctl(p.replace(circles=moved))
    h_x0 = torch.tensor(np.asarray(p.x0, dtype=np.float32))
    h_v0 = torch.tensor(np.asarray(p.v, dtype=np.float32))
    va = h_v0.clone(); a.step_host(h_x0, va, 7)              # captures a's graph on the old environment
    a.set_env(circles=moved)
    va = h_v0.clone(); a.step_host(h_x0, va, 7)              # must re-capture
    vb = h_v0.clone(); b.step_host(h_x0, vb, 7)
    assert torch.equal(va, vb)
    old = h_v0.clone(); _ctl(p).step_host(h_x0, old, 7)
    assert not torch.equal(old, va)
    # a second call replays the captured graph with a new iteration and new inputs
    va2, vb2 = va.clone(), vb.clone()
    a.step_host(h_x0, va2, 8); b.step(b.tensor(p.x0), (d := b.tensor(vb2.numpy())), 8)
    torch.cuda.synchronize()
    assert np.array_equal(va2.numpy(), d.cpu().numpy())
    # timed steps (plain launches) == untimed steps (update kernel as a programmatic dependent of the rollout kernel)
    d1, d2 = b.tensor(p.v), b.tensor(p.v)
    b.step(b.tensor(p.x0), d1, 3)
    b.enable_kernel_timing(True)
    b.step(b.tensor(p.x0), d2, 3)
    assert b.last_rollout_ms() > 0
    vt = h_v0.clone(); b.step_host(h_x0, vt, 3)              # timing on: the call-by-call path
    b.enable_kernel_timing(False)
    torch.cuda.synchronize()
    assert torch.equal(d1, d2) and np.array_equal(vt.numpy(), d1.cpu().numpy())
    a.close(); b.close()
