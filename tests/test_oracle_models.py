"""Pins for the oracle's dynamics and cost functions (no GPU).

Dynamics (1) PAPER.md:29 read as forward Euler (G15); costs per BASELINE configs.
The RK4 integrator and the continuous-time right-hand sides below are written here,
separately from oracle/, to check the Euler order and steady states.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import workloads as W


def test_bicycle_straight_line_closed_form():
    p = W.config0()
    orc = O.Oracle(p)
    X0, Y0, psi, v0 = 1.0, 2.0, 0.3, 2.0
    a, T, dt = 1.5, 20, p.dt
    x = np.array([X0, Y0, psi, v0])
    for _ in range(T):
        x = orc.dynamics(x, [0.0, a])
    # Euler sum: X_T = X_0 + dt cos(psi) (T v0 + dt a T(T-1)/2)
    s = dt * (T * v0 + dt * a * T * (T - 1) / 2)
    assert x[0] == pytest.approx(X0 + math.cos(psi) * s, rel=1e-13)
    assert x[1] == pytest.approx(Y0 + math.sin(psi) * s, rel=1e-13)
    assert x[2] == pytest.approx(psi, abs=1e-15)
    assert x[3] == pytest.approx(v0 + T * dt * a, rel=1e-13)


def test_bicycle_single_step_and_clamps():
    p = W.config0()
    orc = O.Oracle(p)
    x = np.array([0.0, 0.0, math.pi / 2, 2.0])
    xn = orc.dynamics(x, [0.2, 1.0])
    assert xn[0] == pytest.approx(0.0, abs=1e-16 * 10)
    assert xn[1] == pytest.approx(0.05 * 2.0)
    assert xn[2] == pytest.approx(math.pi / 2 + 0.05 * 2.0 * math.tan(0.2) / 0.33)
    assert xn[3] == pytest.approx(2.05)
    # clamps act inside F: steer +-0.35, accel +-3
    assert np.array_equal(orc.dynamics(x, [5.0, 50.0]), orc.dynamics(x, [0.35, 3.0]))
    assert np.array_equal(orc.dynamics(x, [-5.0, -50.0]), orc.dynamics(x, [-0.35, -3.0]))


def _st_rhs(x, delta, Fx, m=4.0, Iz=0.05, lf=0.17, lr=0.17, Cf=30.0, Cr=30.0):
    X, Y, psi, vx, vy, r = x
    af = delta - math.atan2(vy + lf * r, vx)
    ar = -math.atan2(vy - lr * r, vx)
    Fyf, Fyr = Cf * af, Cr * ar
    return np.array([
        vx * math.cos(psi) - vy * math.sin(psi),
        vx * math.sin(psi) + vy * math.cos(psi),
        r,
        (Fx - Fyf * math.sin(delta)) / m + vy * r,
        (Fyf * math.cos(delta) + Fyr) / m - vx * r,
        (lf * Fyf * math.cos(delta) - lr * Fyr) / Iz,
    ])


def _rk4(x, delta, Fx, h, n):
    for _ in range(n):
        k1 = _st_rhs(x, delta, Fx)
        k2 = _st_rhs(x + 0.5 * h * k1, delta, Fx)
        k3 = _st_rhs(x + 0.5 * h * k2, delta, Fx)
        k4 = _st_rhs(x + h * k3, delta, Fx)
        x = x + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    return x


def test_single_track_straight_and_floor():
    p = W.config2()
    orc = O.Oracle(p)
    x = np.array([0.0, 0.0, 0.4, 3.0, 0.0, 0.0])
    for _ in range(60):
        x = orc.dynamics(x, [0.0, 0.0])
    # delta = 0, Fx = 0 keeps vy = r = 0 and a straight line at constant speed
    assert x[4] == 0.0 and x[5] == 0.0 and x[3] == 3.0 and x[2] == 0.4
    assert x[0] == pytest.approx(60 * 0.02 * 3.0 * math.cos(0.4), rel=1e-13)
    assert x[1] == pytest.approx(60 * 0.02 * 3.0 * math.sin(0.4), rel=1e-13)
    # vx floored at 0.5 after the Euler update
    x = np.array([0.0, 0.0, 0.0, 0.52, 0.0, 0.0])
    xn = orc.dynamics(x, [0.0, -10.0])
    assert xn[3] == 0.5


def test_single_track_steady_state_yaw_rate():
    p = W.config2()
    orc = O.Oracle(p)
    delta, vx = 0.02, 2.0
    x = np.array([0.0, 0.0, 0.0, vx, 0.0, 0.0])
    for _ in range(400):
        x = orc.dynamics(x, [delta, 0.0])
    # neutral steer (lf Cf = lr Cr): r -> vx delta / (lf + lr) for small delta
    assert x[5] == pytest.approx(x[3] * delta / 0.34, rel=2e-2)


def test_single_track_euler_is_first_order_vs_rk4():
    p = W.config2()
    x0 = np.array([0.0, 0.0, 0.1, 3.0, 0.1, 0.2])
    delta, Fx, horizon = 0.1, 2.0, 0.4
    ref = _rk4(x0, delta, Fx, 1e-4, int(round(horizon / 1e-4)))
    errs = []
    for dt in (0.02, 0.01, 0.005):
        orc = O.Oracle(p.replace(dt=dt))
        x = x0.copy()
        for _ in range(int(round(horizon / dt))):
            x = orc.dynamics(x, [delta, Fx])
        errs.append(np.abs(x - ref).max())
    assert 1.7 < errs[0] / errs[1] < 2.3 and 1.7 < errs[1] / errs[2] < 2.3


def test_bicycle_euler_is_first_order_vs_rk4():
    def rhs(x, d, a, L=0.33):
        return np.array([x[3] * math.cos(x[2]), x[3] * math.sin(x[2]), x[3] * math.tan(d) / L, a])
    x0 = np.array([0.0, 0.0, 0.2, 2.0]); d, a, horizon = 0.2, 1.0, 1.0
    x = x0.copy(); h = 1e-4
    for _ in range(int(round(horizon / h))):
        k1 = rhs(x, d, a); k2 = rhs(x + 0.5 * h * k1, d, a); k3 = rhs(x + 0.5 * h * k2, d, a); k4 = rhs(x + h * k3, d, a)
        x = x + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    ref = x
    errs = []
    for dt in (0.05, 0.025, 0.0125):
        orc = O.Oracle(W.config0().replace(dt=dt))
        y = x0.copy()
        for _ in range(int(round(horizon / dt))):
            y = orc.dynamics(y, [d, a])
        errs.append(np.abs(y - ref).max())
    assert 1.7 < errs[0] / errs[1] < 2.3 and 1.7 < errs[1] / errs[2] < 2.3


def test_circle_risk_hand_points():
    p = W.config0().replace(circles=np.array([[5.0, 5.0, 0.5], [9.0, 5.0, 0.3]]))
    orc = O.Oracle(p)
    st = lambda X, Y: [X, Y, 0.0, 0.0]
    assert orc.l(st(5.0, 6.0)) == 0.0                      # d = 1.0 > r + margin = 0.7
    assert orc.l(st(5.0, 5.7)) == pytest.approx(0.0, abs=1e-25)  # on the margin circle
    assert orc.l(st(5.0, 5.5)) == pytest.approx(1000 * 0.2**2)   # on the obstacle rim: pen = margin
    assert orc.l(st(5.0, 5.0)) == pytest.approx(1000 * 0.7**2)   # centre: pen = r + margin
    assert orc.l(st(9.0, 5.4)) == pytest.approx(1000 * 0.1**2)   # second circle: 0.3+0.2-0.4
    # both circles contribute (sum over i): point between them with big radii
    p2 = p.replace(circles=np.array([[0.0, 0.0, 2.0], [3.0, 0.0, 2.0]]))
    assert O.Oracle(p2).l(st(1.5, 0.0)) == pytest.approx(2 * 1000 * 0.7**2)
    # hinge margin (test diagnostic): distance to the nearest rim r + 0.2 where l switches between 0 and > 0
    assert orc.hinge_margin(5.0, 6.0) == pytest.approx(0.3) and orc.hinge_margin(5.0, 5.5) == pytest.approx(0.2)
    assert orc.hinge_margin(9.0, 5.4) == pytest.approx(0.1) and orc.hinge_margin(7.0, 5.0) == pytest.approx(1.3)
    r = O.Oracle(W.small(W.config0(near_obstacle=True), K=6, M=5, T=8)).rollout_costs(want_margin=True)
    assert r["margin"].shape == (6, 6) and np.isinf(r["margin"][:, 0]).all() and (r["margin"][:, 1:] > 0).all()


def test_goal_cost_and_terminal():
    p = W.config0()
    orc = O.Oracle(p)
    assert orc.q([18.0, 18.0, 0, 0]) == 0.0
    assert orc.q([1.0, 1.0, 0.785, 2.0]) == pytest.approx(2 * 17.0**2)
    assert orc.phi([1.0, 1.0, 0.785, 2.0]) == pytest.approx(2 * 17.0**2)   # w_phi = 1 (G18)
    assert O.Oracle(p.replace(nom_p=[1.0, 18.0, 18.0, 0.25])).phi([1, 1, 0, 0]) == pytest.approx(0.25 * 578)


def test_ellipse_offset_and_track_cost():
    a, b = 10.0, 6.0
    for th in np.linspace(0, 2 * math.pi, 17):
        assert abs(O.ellipse_offset(a, b, a * math.cos(th), b * math.sin(th))) < 1e-14   # 0 on the centreline
    # first-order agreement with the true normal offset
    for th in (0.3, 1.2, 2.5, 4.0):
        px, py = a * math.cos(th), b * math.sin(th)
        n = np.array([px / a**2, py / b**2]); n /= np.linalg.norm(n)
        for d in (1e-3, -1e-3):
            e = O.ellipse_offset(a, b, px + d * n[0], py + d * n[1])
            assert e == pytest.approx(d, rel=2e-3)
    # on the axes the formula has a closed form: e = (X^2/a^2 - 1) a^2 / (2 |X|)
    assert O.ellipse_offset(a, b, 11.0, 0.0) == pytest.approx((121 / 100 - 1) * 100 / 22)
    assert O.ellipse_offset(a, b, 0.0, 5.0) == pytest.approx((25 / 36 - 1) * 36 / 10)
    p = W.config1()
    orc = O.Oracle(p)
    # q = 5 e^2 + 2 (v-4)^2 + 1000 max(0,|e|-1)^2
    assert orc.q([10.0, 0.0, 1.0, 4.0]) == pytest.approx(0.0, abs=1e-25)
    assert orc.q([10.0, 0.0, 1.0, 3.0]) == pytest.approx(2.0)
    e = O.ellipse_offset(a, b, 11.5, 0.0)
    assert e > 1
    assert orc.q([11.5, 0.0, 0.0, 4.0]) == pytest.approx(5 * e * e + 1000 * (e - 1) ** 2)
    e = O.ellipse_offset(a, b, 0.0, 4.6)
    assert e < -1
    assert orc.q([0.0, 4.6, 0.0, 4.0]) == pytest.approx(5 * e * e + 1000 * (-e - 1) ** 2)
    # single-track: v := vx (component 3)
    p2 = W.config2()
    assert O.Oracle(p2).q([10.0, 0.0, 1.0, 3.0, 9.0, 9.0]) == pytest.approx(2.0)


def test_bilinear_affine_centres_and_clamp():
    h, w, res = 12, 16, 0.5
    iy, ix = np.meshgrid(np.arange(h), np.arange(w), indexing="ij")
    xc, yc = (ix + 0.5) * res, (iy + 0.5) * res
    amap = 2.0 + 0.3 * xc - 0.7 * yc                      # affine in world coordinates
    p = W.config3().replace(costmap=amap, map_res=res, map_ox=0.0, map_oy=0.0, risk_p=[1000.0])
    orc = O.Oracle(p)
    rng = np.random.default_rng(0)
    for _ in range(100):                                  # bilinear reproduces an affine map exactly (interior)
        X = rng.uniform(0.5 * res, (w - 0.5) * res); Y = rng.uniform(0.5 * res, (h - 0.5) * res)
        assert orc.bilinear(X, Y) == pytest.approx(2.0 + 0.3 * X - 0.7 * Y, rel=1e-12)
    rmap = rng.uniform(size=(h, w))
    orc = O.Oracle(p.replace(costmap=rmap))
    for (jy, jx) in [(0, 0), (3, 5), (h - 1, w - 1), (7, 0)]:   # stored values at cell centres; map[row=iy][col=ix]
        assert orc.bilinear((jx + 0.5) * res, (jy + 0.5) * res) == pytest.approx(rmap[jy, jx], rel=1e-13)
    # midpoint of two horizontally adjacent centres
    assert orc.bilinear(3.0 * res, 2.5 * res) == pytest.approx(0.5 * (rmap[2, 2] + rmap[2, 3]), rel=1e-13)
    # clamp-to-edge outside the map
    assert orc.bilinear(-5.0, -5.0) == pytest.approx(rmap[0, 0])
    assert orc.bilinear(1e3, 1e3) == pytest.approx(rmap[h - 1, w - 1])
    assert orc.bilinear(-5.0, (4 + 0.5) * res) == pytest.approx(rmap[4, 0])
    # origin shift
    orc2 = O.Oracle(p.replace(costmap=rmap, map_ox=-2.0, map_oy=1.0))
    assert orc2.bilinear(-2.0 + 2.5 * res, 1.0 + 1.5 * res) == pytest.approx(rmap[1, 2], rel=1e-13)
    # risk = 1000 * cost(p)
    assert orc.l([(5 + 0.5) * res, (3 + 0.5) * res, 0, 0]) == pytest.approx(1000 * rmap[3, 5], rel=1e-13)


def test_scene_generators_match_config_text():
    p0, p1, p2, p3, p4 = W.config0(), W.config1(), W.config2(), W.config3(), W.config4()
    assert p0.circles.shape == (8, 3) and (p0.circles[:, 2] >= 0.3).all() and (p0.circles[:, 2] <= 0.6).all()
    assert p1.circles.shape == (32, 3) and p2.circles.shape == (128, 3) and p4.circles.shape == (64, 3)
    # obstacles lie on the lane: |offset| <= 0.8 (+ first-order distance asymmetry, G25)
    for c in p1.circles:
        assert abs(O.ellipse_offset(10.0, 6.0, c[0], c[1])) < 0.9
    # uniform arc length: consecutive centreline anchor spacing is constant
    px, py, _, _, P = W.ellipse_arclength_points(10.0, 6.0, 32)
    d = np.hypot(np.diff(px), np.diff(py))
    assert d.std() / d.mean() < 0.02 and 51.0 < P < 51.1   # ellipse(10,6) perimeter = 51.05
    assert p3.costmap.shape == (512, 512) and 0.0 <= p3.costmap.min() and p3.costmap.max() <= 1.0
    assert 0.05 < (p3.costmap > 0).mean() < 0.6
    assert p2.nx == 6 and p0.nx == 4
