"""Pins for the oracle's version of the paper's own racing costs (20)-(23), PAPER.md:164-241 (no GPU).

The track is a synthetic rounded rectangle with the published dimensions; the
polyline construction, distances and arc lengths below are written here, independently of oracle/.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _hp():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "paper_hyperparameters.txt")) if l.strip() and not l.startswith("#")]
    return {k: float(v) for k, v in rows}


@pytest.fixture(scope="module")
def prob():
    return W.paper_racing(K=32, M=12, T=30)


@pytest.fixture(scope="module")
def centreline(prob):
    ax, ay, rc = prob.nom_p[:3]
    P = 4 * (ax + ay) + 2 * math.pi * rc
    s = np.linspace(0.0, P, 20001)[:-1]
    pts, P2 = W.rounded_rect_points(ax, ay, rc, s)
    assert P2 == pytest.approx(P)
    return s, pts, P


def test_workload_matches_the_paper_text(prob):
    hp = _hp()
    ax, ay, rc, hw, c1, c2, c3, c4, c5 = prob.nom_p
    assert 4 * (ax + ay) + 2 * math.pi * rc == pytest.approx(hp["centreline_length"], abs=1e-6)
    assert rc == hp["corner_radius"] and 2 * hw == pytest.approx(hp["track_width"])
    assert (c1, c2, c3, c4, c5) == (hp["c1"], hp["c2"], hp["c3"], hp["c4"], hp["c5"])
    assert prob.circles.shape == (int(hp["n_obstacles"]), 3) and np.allclose(prob.circles[:, 2], hp["obstacle_radius"])
    full = W.paper_racing()
    assert (full.K, full.M, full.T) == (int(hp["samples"]), int(hp["realisations"]), int(hp["horizon"]))
    assert full.lam == hp["lambda"] and full.eta == hp["eta"] and full.A == hp["A"]
    assert full.risk == W.RISK_NOMINAL          # l = q


def test_offset_is_distance_to_the_centreline(prob, centreline):
    s, pts, P = centreline
    orc = O.Oracle(prob)
    rng = np.random.default_rng(0)
    for _ in range(300):
        i = int(rng.integers(len(s)))
        d = float(rng.uniform(-0.28, 0.6))
        X, Y = pts[i, 0] + d * pts[i, 2], pts[i, 1] + d * pts[i, 3]
        # brute force: distance to the dense centreline polyline, signed by inside/outside
        dist = np.hypot(pts[:, 0] - X, pts[:, 1] - Y).min()
        assert abs(orc.racing_offset(X, Y)) == pytest.approx(dist, abs=2e-4)
        assert orc.racing_offset(X, Y) == pytest.approx(d, abs=1e-9)
    ax, ay, rc = prob.nom_p[:3]
    assert orc.racing_offset(0.0, 0.0) == pytest.approx(-min(ax, ay) - rc)            # centre of the infield
    assert orc.racing_offset(ax + 1.0, ay + 1.0) == pytest.approx(math.sqrt(2.0) - rc)  # beyond a corner


def test_arclength_projection(prob, centreline):
    s, pts, P = centreline
    orc = O.Oracle(prob)
    # on the centreline s is recovered, and it is insensitive to a lateral offset
    for i in range(0, len(s), 97):
        for d in (0.0, 0.2, -0.2):
            got = orc.racing_arclength(pts[i, 0] + d * pts[i, 2], pts[i, 1] + d * pts[i, 3])
            diff = (got - s[i] + P / 2) % P - P / 2
            assert abs(diff) < 1e-9
    # ds equals the Euclidean step along the centreline
    got = np.array([orc.racing_arclength(x, y) for x, y in pts[::50, :2]])
    step = np.hypot(np.diff(pts[::50, 0]), np.diff(pts[::50, 1]))
    ds = np.diff(got)
    assert np.allclose(ds[ds > -1.0], step[ds > -1.0], rtol=2e-3)      # (the wrap from P to 0 excluded)


def test_boundary_obstacle_and_deviation_costs(prob):
    orc = O.Oracle(prob)
    ax, ay, rc, hw, c1, c2, c3, c4, c5 = prob.nom_p
    free = prob.replace(circles=np.zeros((0, 3)))
    of = O.Oracle(free)
    on_centre = [0.0, -(ay + rc), 0.0, 1.0]
    # (21): d = hw on the centreline -> c1 (atan(-100 hw)/pi + 1/2)
    assert of.q(on_centre) == pytest.approx(c1 * (math.atan(-100 * hw) / math.pi + 0.5), rel=1e-12)
    # on a boundary d = 0 -> mu = 1/2 ; far off the track mu -> 1 ; (21) is >= 0 everywhere
    assert of.q([0.0, -(ay + rc + hw), 0, 0]) == pytest.approx(c1 * 0.5 + c3 * hw**2, rel=1e-12)
    assert of.q([0.0, -(ay + rc + 5.0), 0, 0]) == pytest.approx(c1 * (math.atan(100 * 4.7) / math.pi + 0.5) + c3 * 25.0, rel=1e-12)
    # lateral deviation term c3 e^2, symmetric inside/outside
    for e in (0.1, -0.1):
        want = c1 * (math.atan(-100 * (hw - 0.1)) / math.pi + 0.5) + c3 * 0.01
        assert of.q([0.3, -(ay + rc + e), 0, 0]) == pytest.approx(want, rel=1e-12)
    # (22): indicator, strict inequality, one unit per obstacle
    cx, cy, r = prob.circles[0]
    inside, outside = [cx + 0.5 * r, cy, 0, 0], [cx + 1.0001 * r, cy, 0, 0]
    assert orc.q(inside) - of.q(inside) == pytest.approx(c2)
    assert orc.q(outside) - of.q(outside) == 0.0
    two = prob.replace(circles=np.array([[0.0, -1.0, 0.1], [0.05, -1.0, 0.1]]))
    assert O.Oracle(two).q([0.02, -1.0, 0, 0]) - of.q([0.02, -1.0, 0, 0]) == pytest.approx(2 * c2)
    assert orc.indicator_margin(cx + 0.5 * r, cy) == pytest.approx(0.5 * r)
    # l = q
    assert orc.l(inside) == orc.q(inside) and orc.l(on_centre) == orc.q(on_centre)


def test_progress_terminal_cost(prob):
    orc = O.Oracle(prob)
    ax, ay, rc, hw, c1, c2, c3, c4, c5 = prob.nom_p
    x0 = np.array([0.0, -(ay + rc), 0.0, 1.0])
    # (23): phi = c4 - c5 s, s = distance travelled along the centreline (counter-clockwise positive)
    assert orc.phi(x0, x0) == pytest.approx(c4)
    assert orc.phi([0.25, -(ay + rc) + 0.1, 0, 0], x0) == pytest.approx(c4 - c5 * 0.25)
    assert orc.phi([-0.1, -(ay + rc), 0, 0], x0) == pytest.approx(c4 + c5 * 0.1)       # driving backwards is penalised
    assert orc.phi([c4 / c5, -(ay + rc), 0, 0], x0) == pytest.approx(0.0, abs=1e-12)   # "phi >= 0" up to s = c4/c5
    # across the s = 0 seam (X > 0, Y = 0) the wrapped difference is continuous
    a, b = np.array([ax + rc, -0.05, 0, 0]), np.array([ax + rc, 0.07, 0, 0])
    assert orc.phi(b, a) == pytest.approx(c4 - c5 * 0.12)


def test_iteration_with_l_equal_q(prob):
    p = prob.replace(v=W.random_mean_control(prob, 2, (0.1, 0.5)))
    orc = O.Oracle(p)
    r = orc.rollout_costs(want_margin=True)
    # sigma_w = 0: every noisy rollout is the nominal one and L = sum_t q(x_t) = S - control terms - phi
    p0 = p.replace(sigma_w=[0.0] * 4, gamma=0.0)
    o0 = O.Oracle(p0)
    r0 = o0.rollout_costs()
    for k in (0, 5, 31):
        assert np.allclose(r0["L"][k], r0["L"][k, 0])
        assert r0["S"][k] == pytest.approx(r0["L"][k, 0] + o0.phi(r0["x_nom"][k]), rel=1e-12)
    # margins: col 0 nominal, 1..M noisy, all non-negative and finite on a scene with obstacles
    assert r["margin"].shape == (p.K, p.M + 1) and (r["margin"] >= 0).all() and np.isfinite(r["margin"]).all()
    # eta = 0.2: the last 20 % of the samples are zero-mean
    K0 = math.ceil(0.8 * p.K)
    rz = O.Oracle(p.replace(eta=0.0)).rollout_costs()
    assert np.array_equal(r["u"][:K0], rz["u"][:K0]) and not np.array_equal(r["u"][K0:], rz["u"][K0:])
