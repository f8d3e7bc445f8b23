"""K-sharded step on one GPU: two contexts stand in for two ranks (no kernel waits on another, so this is safe
on a single device); their partials are combined by the library and compared with the unsharded step and the oracle."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2209_12842_b200 import sharded
from paper_2209_12842_b200 import workloads as W
from paper_2209_12842_b200.controller import RaMppi
from parity_utils import TOL_V_ABS, assert_costs_close

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    assert torch.cuda.is_available()
    from paper_2209_12842_b200 import build
    build.build()
    return torch


def _problem(lam):
    p = W.small(W.config1(), K=203, M=64, T=40)
    return p.replace(v=W.random_mean_control(p, 3), lam=lam, eta=0.25)


@pytest.mark.parametrize("world,lam", [(2, 200.0), (3, 200.0), (2, 0.5)])
def test_sharded_step_equals_unsharded(torch_cuda, world, lam):
    p = _problem(lam)
    full = RaMppi(p, 0)
    d_x0, d_v = full.tensor(p.x0), full.tensor(p.v)
    g_full = full.rollout_costs(d_x0, d_v, iteration=7)
    v_ref = d_v.clone()
    full.step(d_x0, v_ref, iteration=7)
    parts, shards = [], []
    for r in range(world):
        sp = sharded.shard_problem(p, world, r)
        ctl = RaMppi(sp, 0)
        shards.append(ctl)
        # the shard's rows are the unsharded rows bit for bit: counters and the eta split use the global k
        g = ctl.rollout_costs(d_x0, d_v, iteration=7)
        sl = slice(sp.k_offset, sp.k_offset + sp.K)
        for key in ("u", "S", "cvar", "S_tilde", "L", "xT"):
            assert torch.equal(g[key], g_full[key][sl]), key
        parts.append(ctl.step_partial(d_x0, d_v, iteration=7).clone())
    d_parts = torch.stack(parts).contiguous()
    v_sh = shards[0].combine_partials(d_parts)
    v_sh_perm = shards[-1].combine_partials(d_parts.flip(0).contiguous())
    torch.cuda.synchronize()
    err = float((v_sh - v_ref).abs().max())
    assert err < 2e-6, err                                   # same weights up to fp32 rounding of the rescale
    assert float((v_sh_perm - v_sh).abs().max()) < 2e-6
    # the partials against the oracle's per-shard restatement, from the GPU's own fp64 S~ and u
    _, St = full.costs_f64()
    St, u = St.cpu().numpy(), g_full["u"].cpu().numpy().astype(np.float64)
    for r, ctl in enumerate(shards):
        sp = ctl.problem
        sl = slice(sp.k_offset, sp.k_offset + sp.K)
        ref = O.shard_partial(St[sl], u[sl], p.lam)
        got = parts[r].cpu().numpy()
        assert got[0] == ref[0]                              # beta_g: exact fp64 min
        assert abs(got[1] - ref[1]) <= 1e-5 * ref[1]
        assert np.abs(got[2:] - ref[2:]).max() <= 1e-5 * max(1.0, np.abs(ref[2:]).max())
    v_orc = O.combine_partials(np.stack([x.cpu().numpy() for x in parts]), p.lam, p.u_min, p.u_max)
    assert np.abs(v_sh.cpu().numpy() - v_orc).max() < TOL_V_ABS
    for c in shards + [full]:
        c.close()


def test_sharded_controller_single_process(torch_cuda):
    """ShardedRaMppi without a process group is the unsharded controller."""
    p = _problem(200.0)
    sc = sharded.ShardedRaMppi(p, 0)
    full = RaMppi(p, 0)
    d_x0 = full.tensor(p.x0)
    v_a, v_b = full.tensor(p.v), full.tensor(p.v)
    sc.step(d_x0, v_a, 3)
    full.step(d_x0, v_b, 3)
    torch.cuda.synchronize()
    assert float((v_a - v_b).abs().max()) < 2e-6
    sc.close(); full.close()


def test_shard_validation(torch_cuda):
    from paper_2209_12842_b200 import binding as B
    p = W.config0(K=16)
    for kw in (dict(k_offset=4), dict(K_total=8), dict(k_offset=20, K_total=32), dict(k_offset=-1, K_total=32)):
        with pytest.raises(B.RaMppiError):
            RaMppi(p.replace(**kw), 0)
