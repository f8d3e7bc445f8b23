"""Parity cases through the CHECKED build of the library (pytest -m gpu): the same sources compiled with -DRA_CHECKED, in
which every kernel asserts its own indices (shared-memory regions against the launcher's size, obstacle / key / noise /
costmap / output indices) and traps on a violation.  compute-sanitizer is closed on the GPU pool (SURVEY.md section 5 asks
for memcheck on config 0), so this is the memory-safety evidence: ragged and extreme sizes, every noise kind and mode,
both half-warp layouts, the costmap edges, the closed loop."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import binding as B
from paper_2209_12842_b200 import build as cuda_build
from paper_2209_12842_b200 import workloads as W

from parity_utils import check_rollout_parity, check_update_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def checked(torch_cuda_module):
    lib = B.open_library(cuda_build.build(checked=True))
    old = B._lib
    B._lib = lib                      # every binding call of this module goes to the checked library
    yield lib
    B._lib = old


@pytest.fixture(scope="module")
def torch_cuda_module():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cuda_build.build()
    return torch


def _ctl(p):
    from paper_2209_12842_b200.controller import RaMppi
    return RaMppi(p, device=0)


def _v(p, seed=0):
    return p.replace(v=W.random_mean_control(p, seed, (0.1, 0.5) if p.dyn == W.DYN_BICYCLE else (0.1, 2.0)))


CASES = {
    "C0": lambda: W.config0(near_obstacle=True),
    "ragged-M17": lambda: W.small(W.config0(near_obstacle=True), K=9, M=17, T=5),
    "M300-8warps": lambda: W.small(W.config4(), K=6, M=300, T=30),
    "M512-T128": lambda: W.small(W.config0(near_obstacle=True), K=3, M=512, T=128),
    "half-4-per-warp": lambda: W.small(W.config4(), K=32771, M=9, T=4),
    "single-track-128-circles": lambda: W.small(W.config2(), K=21, M=128, T=13),
    "costmap-off-the-map": lambda: W.small(W.config3(), K=40, M=128, T=50).replace(x0=np.array([0.2, 25.3, 2.4, 4.0])),
    "materialised-M96": lambda: W.small(W.config1(), K=33, M=96, T=12).replace(noise_mode=W.NOISE_MATERIALISED),
    "materialised-ST-M160": lambda: W.small(W.config2(), K=9, M=160, T=7).replace(noise_mode=W.NOISE_MATERIALISED),
    "jump": lambda: W.small(W.config1(), K=50, M=64, T=21).replace(noise_kind=W.NOISE_JUMP, noise_p=[0.3, 0, 0, 0]),
    "uniform-ST": lambda: W.small(W.config2(), K=11, M=64, T=10).replace(noise_kind=W.NOISE_UNIFORM),
    "racing-l=q": lambda: W.paper_racing(K=24, M=300, T=30),
    "1024-circles": lambda: W.small(W.config1(), K=16, M=64, T=10).replace(
        circles=W.random_circles(np.random.default_rng(9), 1024, 0.1, 0.3, -12.0, 12.0)),
}


@pytest.mark.parametrize("name", list(CASES))
def test_checked_build_parity(checked, torch_cuda_module, name):
    p = _v(CASES[name]())
    ctl, orc = _ctl(p), O.Oracle(p)
    if p.nominal == W.NOM_RACING:         # indicator ties need the margin-aware comparison of test_gpu_parity; here: runs clean
        d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(p.v)
        ctl.rollout_costs(d_x0, d_v, 1)
        ctl.step(d_x0, d_v, 1)
        torch_cuda_module.cuda.synchronize()
    else:
        g, r = check_rollout_parity(p, ctl, orc, iteration=2)
        check_update_parity(p, ctl, orc, r)
        d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(p.v)
        ctl.step(d_x0, d_v, 2)
        torch_cuda_module.cuda.synchronize()
    ctl.close()


def test_checked_build_closed_loop_and_host_step(checked, torch_cuda_module):
    torch = torch_cuda_module
    p = W.small(W.config4(), K=4100, M=64, T=50)          # three sample ranges in the update kernel, its last CTA runs the plant
    ctl = _ctl(p)
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    log, ms = ctl.closed_loop(d_x0, d_v, 0, 12)
    h_x0 = torch.tensor(np.asarray(p.x0, dtype=np.float32))
    h_v = torch.zeros(p.T, 2)
    ctl.step_host(h_x0, h_v, 3)
    ctl.step_host(h_x0, h_v, 4)
    torch.cuda.synchronize()
    assert np.isfinite(log.cpu().numpy()).all() and np.isfinite(h_v.numpy()).all()
    ctl.close()
