"""Pins for the oracle's full iteration: invariants and special cases (no GPU).

PAPER.md Alg.1 :167-223, (3)-(5) :47-57, (14)-(17) :120-136.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _gauss_cvar(alpha):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "gaussian_cvar.txt")) if not l.startswith("#")]
    return {float(a): float(v) for a, v in rows}[alpha]


def _small(p=None, K=48, M=16, T=12):
    p = W.config0(near_obstacle=True) if p is None else p
    p = W.small(p, K, M, T)
    return p.replace(v=W.random_mean_control(p, 0))


def test_weights_invariants_and_shift_invariance():
    p = _small()
    orc = O.Oracle(p)
    r = orc.rollout_costs()
    wu = orc.weights_update(r["S_tilde"], r["u"])
    w = wu["w"] / wu["Z"]
    assert w.sum() == pytest.approx(1.0, rel=1e-14)
    assert 1.0 <= wu["Z"] <= p.K and wu["w"].max() == 1.0           # the argmin has weight exactly 1 (G20)
    assert wu["beta"] == r["S_tilde"].min()
    # "prevent numerical overflow while keeping the solution the same" PAPER.md:57
    wu2 = orc.weights_update(r["S_tilde"] + 12345.0, r["u"])
    assert np.allclose(wu2["v_plus"], wu["v_plus"], atol=1e-9)
    # (4) PAPER.md:51 as a plain weighted mean, clamped (G16)
    vp = np.clip(np.einsum("k,kti->ti", w, r["u"]), p.u_min, p.u_max)
    assert np.allclose(wu["v_plus"], vp, atol=1e-13)


def test_lambda_limits():
    p = _small()
    r = O.Oracle(p).rollout_costs()
    k_star = int(np.argmin(r["S_tilde"]))
    lo = O.Oracle(p.replace(lam=1e-6)).weights_update(r["S_tilde"], r["u"])
    assert np.allclose(lo["v_plus"], np.clip(r["u"][k_star], p.u_min, p.u_max), atol=1e-12)
    hi = O.Oracle(p.replace(lam=1e12)).weights_update(r["S_tilde"], r["u"])
    assert np.allclose(hi["v_plus"], np.clip(r["u"].mean(axis=0), p.u_min, p.u_max), atol=1e-6)


def test_step_equals_stages():
    p = _small()
    orc = O.Oracle(p)
    r = orc.rollout_costs()
    assert np.array_equal(orc.step(), orc.weights_update(r["S_tilde"], r["u"])["v_plus"])
    # threads change nothing (every k independent)
    r4 = orc.rollout_costs(n_threads=4)
    for key in ("u", "S", "cvar", "S_tilde", "L", "xT"):
        assert np.array_equal(r[key], r4[key])
    # k-range evaluation equals the slice
    rs = orc.rollout_costs(k_begin=5, k_end=9)
    assert np.array_equal(rs["S_tilde"], r["S_tilde"][5:9]) and np.array_equal(rs["L"], r["L"][5:9])


def test_soft_filter_and_A_zero_is_mppi():
    p = _small()
    r = O.Oracle(p).rollout_costs()
    assert (r["cvar"] > 0).mean() > 0.2, "risk path not exercised"
    exp = r["S"] + np.where(r["cvar"] > p.C_u, p.A * r["cvar"], 0.0)
    assert np.array_equal(r["S_tilde"], exp)
    # strict threshold (15) PAPER.md:124 and no else branch (G10)
    cu = float(np.median(r["cvar"][r["cvar"] > 0]))
    r2 = O.Oracle(p.replace(C_u=cu, A=10.0)).rollout_costs()
    assert np.array_equal(r2["S_tilde"], r2["S"] + np.where(r2["cvar"] > cu, 10.0 * r2["cvar"], 0.0))
    assert np.array_equal(r2["S_tilde"][r2["cvar"] == cu], r2["S"][r2["cvar"] == cu])
    # A = 0 -> plain MPPI costs (3)
    r0 = O.Oracle(p.replace(A=0.0)).rollout_costs()
    assert np.array_equal(r0["S_tilde"], r0["S"]) and np.array_equal(r0["S"], r["S"])


def test_nominal_cost_formula_and_eta():
    p = _small().replace(eta=0.25, gamma=0.7)
    orc = O.Oracle(p)
    r = orc.rollout_costs()
    K0 = math.ceil(0.75 * p.K)
    # u - v is the same noise for k<K0; zero-mean samples use u = eps (Alg.1 l.8/l.10)
    pe = p.replace(eta=0.0)
    re = O.Oracle(pe).rollout_costs()
    assert np.array_equal(r["u"][:K0], re["u"][:K0])
    assert np.allclose(r["u"][K0:], re["u"][K0:] - p.v[None], atol=1e-15)
    # S_k recomputed from public pieces: sum_t q(x_t) + gamma v^T Sigma^-1 u + phi(x_T)  (3) PAPER.md:47
    for k in (0, K0 - 1, K0, p.K - 1):
        x = np.array(p.x0, dtype=float); S = 0.0
        for t in range(p.T):
            S += orc.q(x) + p.gamma * sum(p.v[t, i] * r["u"][k, t, i] / p.sigma_eps[i] ** 2 for i in range(2))
            x = orc.dynamics(x, r["u"][k, t])
        S += orc.phi(x)
        assert r["S"][k] == pytest.approx(S, rel=1e-13)
        assert np.allclose(r["x_nom"][k], x, atol=1e-13)


def test_zero_dynamics_noise_reproduces_deterministic_rollout():
    p = _small().replace(sigma_w=[0.0] * 4)
    r = O.Oracle(p).rollout_costs()
    # all M rollouts equal the nominal one; CVaR_k = L_k
    assert np.array_equal(r["xT"], np.repeat(r["x_nom"][:, None, :], p.M, axis=1))
    assert np.array_equal(r["L"], np.repeat(r["L"][:, :1], p.M, axis=1))
    assert np.allclose(r["cvar"], r["L"][:, 0], rtol=1e-14)


def test_M1_and_K1():
    p = _small(M=1)
    r = O.Oracle(p).rollout_costs()
    assert np.array_equal(r["cvar"], r["L"][:, 0])
    p1 = _small(K=1)
    orc = O.Oracle(p1)
    r1 = orc.rollout_costs()
    assert np.allclose(orc.step(), np.clip(r1["u"][0], p1.u_min, p1.u_max), atol=1e-15)


def test_risk_cost_sums_pre_step_states():
    # (9) PAPER.md:93: L = sum_{t=0}^{T-1} l(x_t); the last transition does not feed L (G17).
    p = _small(K=4, M=3, T=5)
    orc = O.Oracle(p)
    r = orc.rollout_costs()
    for k in range(p.K):
        for m in range(p.M):
            x = np.array(p.x0, dtype=float); L = 0.0
            for t in range(p.T):
                L += orc.l(x)
                x = orc.dynamics(x, r["u"][k, t]) + orc.state_noise(k, m, t, 1, 0)
            assert r["L"][k, m] == pytest.approx(L, rel=1e-13, abs=1e-13)
            assert np.allclose(r["xT"][k, m], x, atol=1e-13)


@pytest.mark.parametrize("alpha", [0.9, 0.95])
def test_end_to_end_gaussian_cvar_closed_form(alpha):
    """Linear risk l(x)=x[3] on the bicycle with delta=0, eps=0: L is exactly Gaussian.

    v_t = v0 + sum_{s<t}(dt a_s + w_s) so L = sum_{t<T} v_t = T v0 + sum_{s=0}^{T-2} (T-1-s)(dt a_s + w_s):
    mean T v0 + dt sum (T-1-s) a_s, variance sigma_v^2 (T-1)T(2T-1)/6, hence
    CVaR_alpha = mu + sigma pdf(ppf(alpha))/(1-alpha)  (north_star closed form).
    """
    T, M, v0, sv = 12, 1 << 15, 2.0, 0.05
    a = np.linspace(-1.0, 2.0, T)
    p = W.config0().replace(K=2, M=M, T=T, sigma_eps=[0.0, 0.0], sigma_w=[0.02, 0.02, 0.01, sv],
                            risk=W.RISK_LINEAR_STATE, risk_p=[1.0, 3.0], alpha=alpha,
                            v=np.stack([np.zeros(T), a], axis=1), x0=np.array([1.0, 1.0, 0.785, v0]))
    r = O.Oracle(p).rollout_costs(want_xT=False, n_threads=4)
    mu = T * v0 + p.dt * sum((T - 1 - s) * a[s] for s in range(T - 1))
    sigma = sv * math.sqrt((T - 1) * T * (2 * T - 1) / 6)
    closed = mu + sigma * _gauss_cvar(alpha)
    k_tail = O.tail_count(alpha, M)
    mc = 4 * sigma * 2.5 / math.sqrt(k_tail) / 2
    assert abs(r["cvar"][0] - closed) < mc and abs(r["cvar"][1] - closed) < mc
    assert r["L"].mean() == pytest.approx(mu, abs=4 * sigma / math.sqrt(2 * M))
    assert r["L"].std() == pytest.approx(sigma, rel=0.02)
    # sigma_eps = 0: the control-cost term is skipped, u = v exactly
    assert np.array_equal(r["u"][0], p.v)


def test_plant_and_shift():
    p = _small()
    orc = O.Oracle(p)
    x = orc.plant_step(p.x0, [0.1, 1.0], 7)
    assert np.allclose(x, orc.dynamics(p.x0, [0.1, 1.0]) + orc.state_noise(0, 0, 0, 2, 7), atol=0)
    v = np.arange(10.0).reshape(5, 2)
    assert np.array_equal(O.shift(v), np.array([[2, 3], [4, 5], [6, 7], [8, 9], [8, 9.0]]))


def test_eps_draw_scale_layout_and_moments():
    """O1a, the control perturbation eps^k_t ~ N(0, Sigma_eps) (2c) PAPER.md:42, Alg.1 l.4/8 PAPER.md:179-186.

    Pins (a) the scale: std(u - v) per component equals sigma_eps[i] with DISTINCT sigmas (a swap, a sigma^2 or a
    missing factor fails), mean 0, components and steps uncorrelated; (b) the layout of DESIGN.md "RNG layout":
    u[k,t] = v[t] + sigma_eps (.) box_muller(r0, r1) of philox(counter(k, m = 0, t, stream EPS, iteration)), written
    with the oracle's FREE functions (each pinned on its own in test_oracle_rng.py), words (r2, r3) unused."""
    it = 5
    p = W.config0(K=8192, M=1, T=20).replace(seed=0x1234ABCD5678EF01)
    p = p.replace(v=W.random_mean_control(p, 3))
    assert p.sigma_eps[0] != p.sigma_eps[1] and np.abs(p.v).min() > 0
    r = O.Oracle(p).rollout_costs(iteration=it, want_L=False, want_xT=False, n_threads=4)
    d = r["u"] - p.v[None]                                   # [K, T, 2]
    n = p.K * p.T
    for i in range(2):
        s = p.sigma_eps[i]
        assert abs(d[..., i].mean()) < 4 * s / math.sqrt(n)
        assert abs(d[..., i].std() / s - 1.0) < 4 / math.sqrt(2 * n)
        assert abs(((d[..., i] / s) ** 4).mean() - 3.0) < 4 * math.sqrt(96 / n)
    z = d / np.asarray(p.sigma_eps)
    assert abs((z[..., 0] * z[..., 1]).mean()) < 4 / math.sqrt(n)              # the two components of one draw
    assert abs((z[:, :-1, :] * z[:, 1:, :]).mean()) < 4 / math.sqrt(2 * n)     # consecutive steps
    assert abs((z[:-1] * z[1:]).mean()) < 4 / math.sqrt(2 * n)                 # consecutive samples
    # layout, bit for bit
    key = (p.seed & 0xFFFFFFFF, p.seed >> 32)
    rng = np.random.default_rng(0)
    picks = [(0, 0), (p.K - 1, p.T - 1)] + [(int(k), int(t)) for k, t in
                                            zip(rng.integers(0, p.K, 200), rng.integers(0, p.T, 200))]
    for k, t in picks:
        w = O.philox4x32_10(O.counter(k, 0, t, 1, 0, 0, it), key)
        zz = O.box_muller(w[0], w[1])
        for i in range(2):
            assert r["u"][k, t, i] == p.v[t, i] + p.sigma_eps[i] * zz[i]
        other = O.box_muller(w[2], w[3])                      # the unused half of the call is really unused
        assert r["u"][k, t, 0] != p.v[t, 0] + p.sigma_eps[0] * other[0]
    # a different iteration is a different draw; eta's zero-mean samples take the same eps without v
    r0 = O.Oracle(p).rollout_costs(iteration=0, want_L=False, want_xT=False, n_threads=4)
    assert not np.array_equal(r0["u"], r["u"])
