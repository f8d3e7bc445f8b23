"""GPU-vs-oracle parity through the C ABI (run on the B200 box: pytest -m gpu).

Stage-wise, as SURVEY.md section 8(c) lays out: Philox words bit-exact, normals to a few ulp,
states at t=T within 1e-3, costs within 1e-4 relative, CVaR select isolated, update isolated,
then end to end.  Sizes span several CTAs and ragged tails; the oracle finishes in seconds.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import workloads as W

from parity_utils import (TOL_STATE_ABS, assert_costs_close, check_rollout_parity, check_step_parity,
                          check_update_parity, gpu_outputs)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2209_12842_b200 import build
    build.build()
    return torch


def _ctl(p):
    from paper_2209_12842_b200.controller import RaMppi
    return RaMppi(p, device=0)


def _with_v(p, seed=0):
    scale = (0.1, 0.5) if p.dyn == W.DYN_BICYCLE else (0.1, 2.0)
    return p.replace(v=W.random_mean_control(p, seed, scale))


# ------------------------------------------------------------------ RNG
def test_philox_words_bit_exact(torch_cuda):
    torch = torch_cuda
    p = W.config0().replace(seed=0x0123456789ABCDEF)
    ctl = _ctl(p)
    rng = np.random.default_rng(5)
    rows = [O.counter(k, m, t, J, j, s, it) for s in (0, 1, 2) for J in (1, 2) for j in range(J)
            for (k, m, t, it) in [(0, 0, 0, 0), (255, 15, 19, 1), (65535, 255, 127, 499), (7, 300, 59, 2**28 - 1)]]
    rows += [list(rng.integers(0, 2**32, size=4)) for _ in range(2000)]
    ctr = torch.tensor(np.array(rows, dtype=np.int64))
    out = ctl.philox(ctr).cpu().numpy()
    key = (p.seed & 0xFFFFFFFF, p.seed >> 32)
    for r, o in zip(rows, out):
        assert O.philox4x32_10(r, key) == [int(x) for x in o]


@pytest.mark.parametrize("cfg", ["C0", "C2", "uniform", "jump"])
def test_state_noise_draws(torch_cuda, cfg):
    torch = torch_cuda
    p = {"C0": W.config0(), "C2": W.config2(K=64),
         "uniform": W.config0().replace(noise_kind=W.NOISE_UNIFORM, sigma_w=[0.2] * 4),
         "jump": W.config0().replace(noise_kind=W.NOISE_JUMP, sigma_w=[0.45] * 4, noise_p=[0.3, 0, 0, 0])}[cfg]
    ctl, orc = _ctl(p), O.Oracle(p)
    rng = np.random.default_rng(1)
    kmt = np.stack([rng.integers(0, 65536, 4000), rng.integers(0, 512, 4000), rng.integers(0, 128, 4000)], 1)
    w = ctl.state_noise(torch.tensor(kmt), iteration=3).cpu().numpy()
    ref = np.array([orc.state_noise(int(k), int(m), int(t), 1, 3) for k, m, t in kmt])
    sig = np.asarray(p.sigma_w)[: p.nx]
    z, zr = w / sig, ref / sig
    if cfg == "uniform":
        assert np.abs(z - zr).max() < 2e-7            # exact uniforms, one rounding
    elif cfg == "jump":
        assert np.abs(z - zr).max() < 2e-5            # unit direction through the fast normals
        assert np.array_equal(z == 0, zr == 0)        # same trigger decisions (exact uniform compare)
    else:
        # MUFU-based Box-Muller: |dz| <= 4e-6 max(1,|z|) + 4e-7 / max(rho, 1e-3)
        rho = np.sqrt((zr.reshape(len(zr), -1, 2) ** 2).sum(-1, keepdims=True)).repeat(2, -1).reshape(zr.shape)
        bound = 4e-6 * np.maximum(1.0, np.abs(zr)) + 4e-7 / np.maximum(rho, 1e-3)
        assert (np.abs(z - zr) <= bound).all(), (np.abs(z - zr) / bound).max()
        print(f"{cfg}: max |dz| = {np.abs(z - zr).max():.2e}, max |dz|/bound = {(np.abs(z - zr) / bound).max():.2f}")


# ------------------------------------------------------------------ rollouts, costs, CVaR, update
CASES = {
    "C0-near": lambda: W.config0(K=256, M=16, T=20, near_obstacle=True),          # config 0 itself (+ obstacle ahead)
    "C0": lambda: W.config0(),                                                    # config 0 verbatim, v = 0
    "C1-small": lambda: W.small(W.config1(), K=203, M=64, T=40),                  # ragged K, two per lane
    "C2-small": lambda: W.small(W.config2(), K=77, M=128, T=60),                  # single-track, 4 per lane
    "C3-small": lambda: W.small(W.config3(), K=129, M=128, T=50),                 # costmap
    "C4-M16": lambda: W.small(W.config4(), K=101, M=16, T=50),                    # half-warp, odd K
    "C4-M256": lambda: W.small(W.config4(), K=40, M=256, T=50),                   # 8 per lane, two chunks
}


@pytest.mark.parametrize("name", list(CASES))
def test_rollout_costs_cvar_update(torch_cuda, name):
    p = CASES[name]()
    if name != "C0":
        p = _with_v(p)
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc)
    if name == "C0":
        # non-degeneracy report (SURVEY: config 0's random scene usually has no obstacle in reach)
        print(f"{name}: fraction of samples with CVaR>0 = {(r['cvar'] > 0).mean():.3f}")
    else:
        assert (r["cvar"] > 0).mean() > 0.05, "risk path not exercised"
    check_update_parity(p, ctl, orc, r)
    verdict, err = check_step_parity(p, ctl, orc, r)
    print(f"{name}: end-to-end v+ {verdict}, max abs err {err:.2e}")
    ctl.close()


@pytest.mark.parametrize("iteration", [1, 499, 2**28 + 5])
def test_iteration_enters_the_counter(torch_cuda, iteration):
    p = _with_v(W.config0(K=64, near_obstacle=True))
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc, iteration=iteration)
    g0 = gpu_outputs(ctl, p, 0)
    assert not np.array_equal(g0["u"], g["u"])


# ------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("K,M,T", [(1, 1, 1), (3, 1, 7), (5, 2, 3), (9, 17, 5), (33, 20, 9), (17, 50, 11),
                                    (6, 300, 30), (4, 512, 8), (2, 96, 128), (31, 33, 2),
                                    (32771, 9, 6), (32769, 16, 3)])   # M <= 16 with four samples per warp (K >= 32768), ragged K
def test_ragged_and_extreme_sizes(torch_cuda, K, M, T):
    p = W.small(W.config0(near_obstacle=True), K=K, M=M, T=T)
    p = _with_v(p.replace(sigma_w=[0.05, 0.05, 0.02, 0.1]))
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc)
    check_update_parity(p, ctl, orc, r)
    ctl.close()


def test_paper_sized_workload_M300(torch_cuda):
    """The paper's own sizes: 1024 samples x 300 realisations, T=30, lambda=0.35, eta=0.2, A=10
    (tests/golden/paper_hyperparameters.txt); a slice of samples against the oracle."""
    hp = {k: float(v) for k, v in (l.split() for l in open(
        __import__("os").path.join(__import__("os").path.dirname(__file__), "golden", "paper_hyperparameters.txt"))
        if not l.startswith("#"))}
    p = W.config4(K=int(hp["samples"]), M=int(hp["realisations"]), T=int(hp["horizon"]))
    p = _with_v(p.replace(lam=hp["lambda"], gamma=hp["lambda"], eta=hp["eta"], A=hp["A"], alpha=0.9, C_u=0.5, B=2.0))
    ctl, orc = _ctl(p), O.Oracle(p)
    check_rollout_parity(p, ctl, orc, k_begin=800, k_end=864)   # straddles K0 = ceil(0.8 K) = 820
    ctl.close()


def test_parameters_eta_B_Cu_A(torch_cuda):
    base = _with_v(W.small(W.config1(), K=96, M=64, T=20))
    for kw in (dict(eta=0.25), dict(B=3.0), dict(C_u=50.0, A=10.0), dict(A=0.0), dict(gamma=0.0),
               dict(alpha=0.5), dict(alpha=0.99), dict(lam=100.0),
               dict(alpha=0.3)):   # k_tail = 45: the radix selector with two slots per lane
        p = base.replace(**kw)
        ctl, orc = _ctl(p), O.Oracle(p)
        g, r = check_rollout_parity(p, ctl, orc)
        check_update_parity(p, ctl, orc, r)
        if "lam" in kw:   # soft weights: end-to-end v+ must match outright
            verdict, err = check_step_parity(p, ctl, orc, r)
            assert verdict == "match", verdict
        ctl.close()


def test_degenerate_cases(torch_cuda):
    base = _with_v(W.small(W.config0(near_obstacle=True), K=40, M=32, T=12))
    # sigma_w = 0: all M rollouts coincide with the deterministic one, CVaR_k = L_k
    p = base.replace(sigma_w=[0.0] * 4)
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc)
    assert np.array_equal(g["L"], np.repeat(g["L"][:, :1], p.M, 1))
    assert np.allclose(g["cvar"], g["L"][:, 0], rtol=1e-6)
    # empty obstacle set: L == 0 exactly, S~ == S
    p = base.replace(circles=np.zeros((0, 3)))
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc)
    assert not g["L"].any() and not g["cvar"].any() and np.array_equal(g["S"], g["S_tilde"])
    # sigma_eps = 0: u = v exactly, control-cost term skipped, K identical samples -> v+ = clamp(v)
    p = base.replace(sigma_eps=[0.0, 0.0])
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc)
    assert np.array_equal(g["u"], np.repeat(p.v[None].astype(np.float32), p.K, 0))
    verdict, err = check_step_parity(p, ctl, orc, r)
    assert verdict == "match"
    # test-only linear risk with negative values exercises the signed radix keys
    p = base.replace(risk=W.RISK_LINEAR_STATE, risk_p=[-1.0, 3.0])
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc)
    assert (g["cvar"] < 0).all()


def test_non_gaussian_noise_kinds(torch_cuda):
    base = _with_v(W.small(W.config1(), K=64, M=64, T=20))
    for kw in (dict(noise_kind=W.NOISE_UNIFORM, sigma_w=[0.05, 0.05, 0.02, 0.1]),
               dict(noise_kind=W.NOISE_JUMP, sigma_w=[0.45, 0.45, 0.1, 0.3], noise_p=[0.02, 0, 0, 0])):
        p = base.replace(**kw)
        ctl, orc = _ctl(p), O.Oracle(p)
        check_rollout_parity(p, ctl, orc)
        ctl.close()


def test_materialised_noise_equals_fused(torch_cuda):
    # M = 96 / 160: three / five slots of 32 realisations with two interleaved per lane, so the last group carries one
    # slot past the end (its loads must stay inside the noise tensor: ADVICE r1)
    for p in (_with_v(W.small(W.config3(), K=65, M=128, T=10)), _with_v(W.small(W.config2(), K=20, M=50, T=8)),
              _with_v(W.small(W.config1(), K=33, M=96, T=13)), _with_v(W.small(W.config2(), K=9, M=160, T=7)),
              # odd horizons with two words per step: the generator's last Philox call serves one step only
              _with_v(W.small(W.config3(), K=7, M=32, T=5)).replace(noise_kind=W.NOISE_UNIFORM, sigma_w=[0.2] * 4),
              _with_v(W.small(W.config0(near_obstacle=True), K=300, M=16, T=1))):
        a = gpu_outputs(_ctl(p), p)
        b = gpu_outputs(_ctl(p.replace(noise_mode=W.NOISE_MATERIALISED)), p)
        # same draws; the fused kernel contracts sigma*z + x into one FMA, so equality is to rounding
        for k in ("S", "u"):
            assert np.array_equal(a[k], b[k]), k
        assert np.abs(a["xT"] - b["xT"]).max() < 1e-5
        for k in ("cvar", "S_tilde", "L"):
            assert_costs_close(a[k], b[k], k, tol=1e-5)


def test_single_track_floor_and_x0_floor(torch_cuda):
    p = _with_v(W.small(W.config2(), K=24, M=32, T=30))
    p = p.replace(x0=np.array([10.0, 0.0, np.pi / 2, 0.3, 0.0, 0.0], dtype=np.float32).astype(np.float64),
                  v=np.tile(np.array([[0.0, -10.0]]), (30, 1)))
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc)
    assert (g["xT"][..., 3] >= 0.5).all() and (g["xT"][..., 3] == 0.5).any()


@pytest.mark.parametrize("case", ["bicycle-3-turns", "single-track-2-turns", "bicycle-15-turns"])
def test_yaw_winding_at_T128(torch_cuda, case):
    """The noisy rollouts take sin/cos of the yaw with MUFU.SIN/COS on the unreduced angle (the yaw is reduced to
    [-pi, pi) once, at rollout start), so that error grows like 2^-23 |psi| with the winding inside the horizon.  Full
    steering lock held over the longest horizon, T = 128, winds the yaw by 3 turns at config speed, by 15 turns at up to
    25 m/s (far outside any workload), and spins a single-track car: the states at t = T must stay within north_star's
    1e-3 of the oracle's libm sin/cos.  They do with a factor 3 to spare even at 15 turns, and the same library with an
    exactly reduced sin/cos in its place gives the same errors to 10 % (profiles/r3_yaw_winding.md): what limits these
    cases is the fp32 Euler sum of yaw and speed over 128 steps, not the unreduced angle.
    Costs: these scenes score only rim-grazing rollouts (under 1 % of them, L of order 1), where a hinge of 1000 per
    metre squared turns an in-tolerance position error into a relative cost error above 1e-4 whatever sin/cos is used, so
    the cost checks run at 3e-3 here; the 1e-4 cost tolerance is pinned by every other case of this file."""
    from parity_utils import rel_err
    T = 128
    if case.startswith("bicycle"):
        v0, accel, min_turns = (3.0, 0.0, 2.9) if case == "bicycle-3-turns" else (6.0, 3.0, 10.0)
        p = W.small(W.config0(near_obstacle=True), K=40, M=64, T=T)
        p = p.replace(x0=np.array([1.0, 1.0, 3.0, v0]), v=np.tile(np.array([[0.35, accel]]), (T, 1)))
    else:                      # initial yaw rate 12 rad/s, steering at the clamp, noisy yaw rate
        p = W.small(W.config2(), K=40, M=64, T=T)
        p = p.replace(dt=0.05, x0=np.array([10.0, 0.0, np.pi / 2, 4.0, 0.0, 12.0]),
                      v=np.tile(np.array([[0.35, 4.0]]), (T, 1)),
                      sigma_w=[0.01, 0.01, 0.005, 0.05, 0.05, 0.3])
        min_turns = 1.5
    ctl, orc = _ctl(p), O.Oracle(p)
    g, r = check_rollout_parity(p, ctl, orc, tol_cost=3e-3)
    turns = np.abs(r["xT"][..., 2] - p.x0[2]) / (2 * np.pi)
    err = np.abs(g["xT"] - r["xT"]).max(axis=(0, 1))
    print(f"{case}: yaw winding median {np.median(turns):.1f} turns, max {turns.max():.1f}; max |x_T err| per component "
          f"{err}; max rel err of L {rel_err(g['L'], r['L']).max():.2e}, of S {rel_err(g['S'], r['S']).max():.2e}; "
          f"fraction of rollouts with L > 0: {(r['L'] > 0).mean():.3f}")
    assert np.median(turns) > min_turns, "the case does not wind the yaw"
    assert err.max() < TOL_STATE_ABS / 2
    ctl.close()


# ------------------------------------------------------------------ the paper's own racing costs (NEXT row 2)
def _racing_compare(p, g, r, sl):
    """Indicator obstacle cost (22) is a float decision: exclude rollouts whose distance to some
    obstacle rim comes within 3e-6 m of the jump (both answers are then correct), compare the rest."""
    tie = r["margin"] < 3e-6                       # [n, M+1]: col 0 nominal, 1.. noisy
    ok_L = ~tie[:, 1:]
    assert ok_L.mean() > 0.99
    assert np.abs(g["xT"][sl] - r["xT"]).max() < TOL_STATE_ABS
    assert np.abs(g["u"][sl] - r["u"]).max() < 2e-6 * max(1.0, np.abs(r["u"]).max())
    from parity_utils import rel_err
    assert rel_err(g["L"][sl], r["L"])[ok_L].max() < 1e-4
    clean = ~tie.any(axis=1)
    assert clean.mean() > 0.3
    assert rel_err(g["S"][sl], r["S"])[~tie[:, 0]].max() < 1e-4
    assert rel_err(g["cvar"][sl], r["cvar"])[clean].max() < 1e-4
    assert rel_err(g["S_tilde"][sl], r["S_tilde"])[clean].max() < 1e-4
    return clean


def test_paper_racing_costs_l_equals_q(torch_cuda):
    p = W.paper_racing(K=96, M=300, T=30)          # the paper's M = 300: ragged over 32 lanes
    p = p.replace(v=W.random_mean_control(p, 4, (0.1, 0.5)))
    ctl, orc = _ctl(p), O.Oracle(p)
    g = gpu_outputs(ctl, p)
    r = orc.rollout_costs(n_threads=8, want_margin=True)
    clean = _racing_compare(p, g, r, slice(0, p.K))
    assert (r["cvar"] > p.C_u).mean() > 0.05 and (r["L"] > 1.0).mean() > 0.01      # obstacles / boundary are hit
    # CVaR select isolated on the GPU's own L, and the update stage isolated
    k_tail = O.tail_count(p.alpha, p.M)
    iso = np.array([O.cvar_topk(g["L"][i].astype(np.float64), k_tail) for i in range(p.K)])
    assert_costs_close(g["cvar"], iso, "CVaR vs sort of GPU L", tol=2e-6)
    check_update_parity(p, ctl, orc, r)
    if clean.all():
        verdict, err = check_step_parity(p, ctl, orc, r)
        print(f"paper-racing: end-to-end v+ {verdict}")
    ctl.close()


def test_paper_racing_full_size_sampled(torch_cuda):
    p = W.paper_racing()                           # 1024 x 300 x 30 = the paper's 3.072e5 trajectories
    p = p.replace(v=W.random_mean_control(p, 5, (0.1, 0.5)))
    ctl, orc = _ctl(p), O.Oracle(p)
    g = gpu_outputs(ctl, p)
    for kb in (0, 800, p.K - 48):                  # 800..848 straddles K0 = ceil(0.8 K) = 820 (eta = 0.2)
        r = orc.rollout_costs(k_begin=kb, k_end=kb + 48, n_threads=8, want_margin=True)
        _racing_compare(p, g, r, slice(kb, kb + 48))
    ctl.close()


def test_paper_racing_single_track(torch_cuda):
    p = W.paper_racing(K=64, M=96, T=30, single_track=True)
    p = p.replace(v=W.random_mean_control(p, 6, (0.1, 0.2)))
    ctl, orc = _ctl(p), O.Oracle(p)
    g = gpu_outputs(ctl, p)
    r = orc.rollout_costs(n_threads=8, want_margin=True)
    _racing_compare(p, g, r, slice(0, p.K))
    ctl.close()


def test_racing_nominal_cost_with_hinge_circle_risk(torch_cuda):
    """Racing nominal cost (20)-(23) together with the BASELINE hinge risk: the indicator (22) tests the bare radius
    (it has no margin) while the hinge risk tests r + margin, from one obstacle table."""
    p = W.paper_racing(K=64, M=64, T=30)
    p = p.replace(risk=W.RISK_CIRCLES, risk_p=[1000.0, 0.2], v=W.random_mean_control(p, 7, (0.1, 0.5)))
    ctl, orc = _ctl(p), O.Oracle(p)
    g = gpu_outputs(ctl, p)
    r = orc.rollout_costs(n_threads=8, want_margin=True)
    _racing_compare(p, g, r, slice(0, p.K))
    assert (r["L"] > 0).mean() > 0.01 and (r["S"] != r["S"][0]).any()
    ctl.close()


def test_baseline_mppi_mode_skips_the_noisy_rollouts(torch_cuda):
    """A = 0 is the MPPI of section II: S~ = S, and ra_mppi_step needs no noisy rollout."""
    torch = torch_cuda
    p = _with_v(W.small(W.config1(), K=300, M=64, T=25)).replace(A=0.0, lam=50.0)
    ctl, orc = _ctl(p), O.Oracle(p)
    assert ctl.launches_per_step == 3      # sampling, nominal rollout, weights/update
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(p.v)
    ctl.step(d_x0, d_v, 3)
    S64, St64 = ctl.costs_f64()
    torch.cuda.synchronize()
    assert np.array_equal(S64.cpu().numpy(), St64.cpu().numpy())
    ref = orc.step(iteration=3, n_threads=8)
    assert np.abs(d_v.cpu().numpy() - ref).max() < 1e-4
    # the diagnostic call still runs the risk path and reports CVaR, with S~ = S
    g, r = check_rollout_parity(p, ctl, orc, iteration=3)
    assert (g["cvar"] > 0).any() and np.array_equal(g["S"], g["S_tilde"])
    assert _ctl(p.replace(A=1.0)).launches_per_step == 4
    # no rollout kernel is launched by an A = 0 step, so there is nothing to time: a clear error, not a CUDA failure
    from paper_2209_12842_b200 import binding as B
    ctl.enable_kernel_timing(True)
    ctl.step(d_x0, d_v, 4)
    with pytest.raises(B.RaMppiError) as e:
        ctl.last_rollout_ms()
    assert e.value.status == B.RA_EINVAL and "timed" in str(e.value)
    # a diagnostics pass whose risk costs overflow (CVaR = inf) must not leave J_C = 0 * inf = NaN behind in the S~ of the
    # A = 0 steps that follow it (they skip the noisy rollouts and so never rewrite J_C)
    q = p.replace(risk=W.RISK_LINEAR_STATE, risk_p=[3e38, 3.0, 0.0, 0.0])   # weight * speed overflows fp32
    c2 = _ctl(q)
    x, v1, v2 = c2.tensor(q.x0), c2.tensor(q.v), c2.tensor(q.v)
    c2.step(x, v1, 5)
    out = c2.rollout_costs(x, c2.tensor(q.v), 5)
    assert not torch.isfinite(out["cvar"]).all(), "the case does not overflow"
    assert torch.equal(out["S"], out["S_tilde"])
    c2.step(x, v2, 5)
    torch.cuda.synchronize()
    assert torch.isfinite(v2).all() and torch.equal(v1, v2)
    c2.close()


def test_largest_shared_memory_footprint(torch_cuda):
    """M <= 16 with two slots per lane (K >= 32768) at T = 128 and 1024 circles is the rollout kernel's largest CTA
    (32 control-effect rows + keys + circles = 82 KB of shared memory); also reached by set_env on a context created with
    few circles.  Slices of samples against the oracle (first CTA, a middle one, the ragged last one); the step runs."""
    torch = torch_cuda
    p = _with_v(W.small(W.config1(n_obs=1024), K=32768 + 5, M=16, T=128))
    assert p.circles.shape[0] == 1024
    ctl, orc = _ctl(p), O.Oracle(p)
    for k0, k1 in ((0, 24), (20000, 20016), (p.K - 9, p.K)):
        g, r = check_rollout_parity(p, ctl, orc, k_begin=k0, k_end=k1)
    assert (r["cvar"] > 0).mean() > 0.05, "risk path not exercised"
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(p.v)
    ctl.step(d_x0, d_v, 0)
    torch.cuda.synchronize()
    assert torch.isfinite(d_v).all()
    ctl.close()
    few = p.replace(circles=p.circles[:8])
    a = _ctl(few)
    a.set_env(circles=p.circles)
    ga = a.rollout_costs(a.tensor(p.x0), a.tensor(p.v), 0, want_xT=False, want_u=False)
    torch.cuda.synchronize()
    assert np.array_equal(ga["L"].cpu().numpy(), g["L"])
    a.close()


def test_set_env_replaces_obstacles_and_costmap(torch_cuda):
    """ra_mppi_set_env: a context whose environment was replaced equals a fresh context built on the new one."""
    torch = torch_cuda
    from paper_2209_12842_b200 import binding as B
    # obstacles (different count, too)
    p = _with_v(W.small(W.config1(), K=64, M=64, T=20))
    moved = np.concatenate([p.circles[:20] + np.array([0.15, -0.1, 0.05]), [[10.0, 0.5, 0.4]]])
    a, b = _ctl(p), _ctl(p.replace(circles=moved))
    d_x0, d_v = a.tensor(p.x0), a.tensor(p.v)
    before = a.rollout_costs(d_x0, d_v, 2)["S_tilde"].clone()
    a.set_env(circles=moved)
    ga, gb = a.rollout_costs(d_x0, d_v, 2), b.rollout_costs(d_x0, d_v, 2)
    torch.cuda.synchronize()
    for key in ("S", "cvar", "S_tilde", "L", "xT"):
        assert torch.equal(ga[key], gb[key]), key
    assert not torch.equal(before, ga["S_tilde"])
    # the captured closed-loop graph is rebuilt after the change
    xa, va, xb, vb = a.tensor(p.x0), a.tensor(p.v), b.tensor(p.x0), b.tensor(p.v)
    a.closed_loop(xa, va, 0, 3, log=False, timing=False)
    a.set_env(circles=moved)
    xa.copy_(xb); va.copy_(vb)
    a.closed_loop(xa, va, 0, 3, log=False, timing=False)
    b.closed_loop(xb, vb, 0, 3, log=False, timing=False)
    torch.cuda.synchronize()
    assert torch.equal(xa, xb) and torch.equal(va, vb)
    with pytest.raises(B.RaMppiError):
        a.set_env(circles=np.zeros((2000, 3)))
    a.close(); b.close()
    # costmap: same size, new content and origin
    p = _with_v(W.small(W.config3(), K=48, M=32, T=20))
    cm = np.ascontiguousarray(p.costmap[::-1, ::-1])
    a, b = _ctl(p), _ctl(p.replace(costmap=cm, map_ox=-0.3))
    a.set_env(costmap=cm, map_ox=-0.3)
    d_x0, d_v = a.tensor(p.x0), a.tensor(p.v)
    ga, gb = a.rollout_costs(d_x0, d_v, 1), b.rollout_costs(d_x0, d_v, 1)
    torch.cuda.synchronize()
    assert torch.equal(ga["L"], gb["L"]) and torch.equal(ga["S_tilde"], gb["S_tilde"])
    with pytest.raises(B.RaMppiError):
        a.set_env(costmap=cm[:100, :100])
    a.close(); b.close()
