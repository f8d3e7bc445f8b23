"""Seeded random configurations through the whole path against the oracle (sizes, models, costs, noise kinds and
parameters drawn together), to reach combinations the hand-written cases do not name."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import workloads as W

from parity_utils import check_rollout_parity, check_update_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2209_12842_b200 import build
    build.build()
    return torch


def _random_problem(seed):
    rng = np.random.default_rng(7000 + seed)
    base = [W.config1, W.config2, W.config3, lambda: W.config0(near_obstacle=True), lambda: W.config4()][seed % 5]()
    K = int(rng.integers(1, 71))
    M = int(rng.choice([1, 2, 7, 16, 17, 31, 32, 33, 64, 96, 100, 128, 160, 256, 300]))
    T = int(rng.integers(1, 41))
    p = W.small(base, K=K, M=M, T=T)
    scale = (0.1, 0.5) if p.dyn == W.DYN_BICYCLE else (0.1, 2.0)
    kind = int(rng.integers(0, 3))
    alpha = float(np.float32(rng.uniform(0.05, 0.99)))
    if rng.integers(0, 3) == 0 and M >= 2:
        # alpha just below / above a value that makes (1-alpha) M an integer j: the tail count must flip between j and
        # j + 1 on both sides alike (5e-7 M away: outside the library's 2^-23 M guard window, G11)
        j, side = int(rng.integers(1, M)), float(rng.choice([-1.0, 1.0]))
        alpha = float(np.float32(1.0 - (j + side * 5e-7 * M) / M))
    return p.replace(
        v=W.random_mean_control(p, seed, scale), seed=int(rng.integers(0, 2**40)),
        alpha=alpha, eta=float(rng.choice([0.0, 0.3, 0.7, 0.35, 0.9])),
        noise_mode=int(rng.choice([W.NOISE_FUSED, W.NOISE_FUSED, W.NOISE_MATERIALISED])),
        B=float(rng.choice([1.0, 2.5])), A=float(rng.choice([1.0, 5.0])), C_u=float(rng.choice([0.0, 20.0])),
        lam=float(rng.choice([0.5, 50.0])), noise_kind=kind,
        noise_p=[0.3, 0.0, 0.0, 0.0] if kind == W.NOISE_JUMP else [0.0] * 4)


@pytest.mark.parametrize("seed", range(int(__import__("os").environ.get("RA_FUZZ_SEEDS", "20"))))
def test_random_configuration(torch_cuda, seed):
    from paper_2209_12842_b200.controller import RaMppi
    p = _random_problem(seed)
    ctl, orc = RaMppi(p, device=0), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc, iteration=int(seed * 37 + 1))
    check_update_parity(p, ctl, orc, r)
    ctl.close()
