"""The closed-loop RA-MPPI vs MPPI study: bookkeeping on hand-built logs (no GPU) and the
configuration of its arms on the GPU (PAPER.md:247: equal numbers of sampled trajectories; :263: collision definition)."""
import math

import numpy as np
import pytest

from paper_2209_12842_b200 import closed_loop_study as S
from paper_2209_12842_b200 import workloads as W


def _lap_points(p, n_per_lap, laps, offset=0.0):
    """Points on the centreline (+ lateral offset), counter-clockwise, `laps` times round."""
    ax, ay, rc = p.nom_p[:3]
    P = 4 * (ax + ay) + 2 * math.pi * rc
    s = np.arange(int(n_per_lap * laps) + 1) * P / n_per_lap
    pts, _ = W.rounded_rect_points(ax, ay, rc, s % P)
    return pts[:, 0] + offset * pts[:, 2], pts[:, 1] + offset * pts[:, 3]


def _log(X, Y, v=1.0):
    log = np.zeros((len(X), 6), dtype=np.float32)
    log[:, 0], log[:, 1], log[:, 3] = X, Y, v
    return log


def test_track_metrics_counts_laps_and_collision_events():
    p = S.scenario("gaussian").replace(circles=np.array([[1.0, -1.0537 + 0.2, 0.05]]))   # one small obstacle off the line
    X, Y = _lap_points(p, 400, 3.0)
    m = S.track_metrics(p, _log(X, Y, v=2.0))
    assert m["laps"] == pytest.approx(3.0, abs=0.01) and m["collision_events"] == 0 and m["steps_in_collision"] == 0
    assert m["lap_time_s"] == pytest.approx(len(X) * p.dt / 3.0, rel=0.01) and m["mean_speed"] == pytest.approx(2.0)
    # clockwise driving counts as negative laps, normalised by their magnitude
    m = S.track_metrics(p, _log(X[::-1], Y[::-1]))
    assert m["laps"] == pytest.approx(-3.0, abs=0.01) and m["collisions_per_lap"] == 0.0
    # two off-track excursions (each several steps long = one event each) and one pass through an obstacle
    Xo, Yo = X.copy(), Y.copy()
    Xb, Yb = _lap_points(p, 400, 3.0, offset=p.nom_p[3] + 0.05)             # 5 cm beyond the outer boundary
    for a, b in ((100, 110), (700, 720)):
        Xo[a:b], Yo[a:b] = Xb[a:b], Yb[a:b]
    c = np.array([[Xo[50], Yo[50], 0.02]])                                     # an obstacle on the line, 3 steps wide at most
    m = S.track_metrics(p.replace(circles=c), _log(Xo, Yo))
    assert m["off_track_events"] == 2 and m["steps_in_collision"] >= 30
    assert m["obstacle_events"] == 3                                           # the point is passed once per lap
    assert m["collision_events"] == 5 and m["collisions_per_lap"] == pytest.approx(5 / 3.0, rel=0.01)
    # inside the lane edge is fine: 1 cm inside the boundary is no collision ("areas outside of the track")
    Xi, Yi = _lap_points(p, 400, 1.0, offset=-(p.nom_p[3] - 0.01))
    assert S.track_metrics(p.replace(circles=np.zeros((0, 3))), _log(Xi, Yi))["collision_events"] == 0


def test_arms_have_equal_trajectory_counts():
    ra = S.scenario("jump", alpha=0.8, C_u=4.0)
    mp, mk = S.mppi_arm(ra), S.mppi_arm(ra, equal_trajectories=False)
    assert ra.K * ra.M == 307200 == mp.K * mp.M and mp.M == 1 and mp.A == 0.0      # PAPER.md:247, last sentence
    assert mk.K == ra.K and mk.A == 0.0
    assert ra.noise_kind == W.NOISE_JUMP and ra.noise_p[0] == 0.02 and ra.alpha == 0.8 and ra.C_u == 4.0
    assert ra.A == 10.0 and ra.lam == 0.35 and ra.eta == 0.2 and ra.T == 30
    g, u = S.scenario("gaussian"), S.scenario("uniform")
    assert g.sigma_w == u.sigma_w and np.allclose(np.array(ra.sigma_w) / np.array(g.sigma_w), 0.45 / 0.2)


@pytest.mark.gpu
def test_study_arms_on_the_gpu():
    import torch
    assert torch.cuda.is_available()
    from paper_2209_12842_b200 import build
    build.build()
    rows = S.run_arms("gaussian", 0.9, 8.0, iterations=300)
    by = {r["controller"]: r for r in rows}
    assert by["RA-MPPI"]["launches_per_step"] == 4 and by["MPPI"]["launches_per_step"] == 3 == by["MPPI-K"]["launches_per_step"]
    assert by["MPPI"]["K"] == 307200 and by["RA-MPPI"]["K"] * by["RA-MPPI"]["M"] == 307200
    for r in rows:
        assert np.isfinite(r["laps"]) and r["controller_hz"] > 100 and r["mean_speed"] >= 0.2 - 1e-6   # the speed floor holds
