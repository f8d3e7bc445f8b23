"""Seeded synthetic workloads (BASELINE.json configs 0-4) for RA-MPPI.

This module is the one thing the oracle's tests and the CUDA path share: plain
data (a :class:`Problem` record) and scene generators (obstacles, ellipse track,
costmap).  It holds none of the method's arithmetic -- no dynamics, costs, RNG,
CVaR or weights -- and imports neither ``oracle/`` nor the CUDA binding.

The paper (arXiv 2209.12842) measures on a private race track (PAPER.md:251-257,
layout only in a missing figure); BASELINE.json replaces it with the five
synthetic workloads built here.  Scene conventions are DESIGN.md readings
G23-G27.  Scenes are drawn in fp64 from ``numpy.random.default_rng(config index)``
and handed to both sides as identical fp32-representable arrays.
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

DYN_BICYCLE, DYN_SINGLE_TRACK = 0, 1
NOM_GOAL, NOM_ELLIPSE_TRACK, NOM_RACING = 0, 1, 2
RISK_CIRCLES, RISK_COSTMAP, RISK_LINEAR_STATE, RISK_NOMINAL = 0, 1, 2, 3
NOISE_GAUSSIAN, NOISE_UNIFORM, NOISE_JUMP = 0, 1, 2
NOISE_FUSED, NOISE_MATERIALISED = 0, 1


def _f32(a):
    """Round to fp32 and return as fp64 so both sides start from identical reals."""
    return np.asarray(a, dtype=np.float32).astype(np.float64)


@dataclass
class Problem:
    """One RA-MPPI controller-iteration problem (BASELINE letters: K samples, M realisations, T steps)."""

    name: str
    K: int
    M: int
    T: int
    dt: float
    dyn: int
    dyn_p: list
    u_min: list
    u_max: list
    sigma_eps: list
    sigma_w: list
    alpha: float
    lam: float
    gamma: float
    A: float = 1.0
    B: float = 1.0
    C_u: float = 0.0
    eta: float = 0.0
    nominal: int = NOM_GOAL
    nom_p: list = field(default_factory=list)
    risk: int = RISK_CIRCLES
    risk_p: list = field(default_factory=list)
    noise_kind: int = NOISE_GAUSSIAN
    noise_p: list = field(default_factory=lambda: [0.0, 0.0, 0.0, 0.0])
    noise_mode: int = NOISE_FUSED
    seed: int = 0
    x0: np.ndarray = None
    v: np.ndarray = None  # [T,2] mean control sequence
    circles: Optional[np.ndarray] = None  # [n,3] x,y,r
    costmap: Optional[np.ndarray] = None  # [h,w]
    map_res: float = 0.0
    map_ox: float = 0.0
    map_oy: float = 0.0
    k_offset: int = 0   # K-sharding: global index of this shard's first sample
    K_total: int = 0    # K-sharding: samples over all shards (0 = not sharded)

    @property
    def nx(self) -> int:
        return 6 if self.dyn == DYN_SINGLE_TRACK else 4

    @property
    def state_steps(self) -> int:
        return self.K * self.M * self.T

    def replace(self, **kw) -> "Problem":
        return dataclasses.replace(self, **kw)


# --------------------------------------------------------------------------- scenes
def random_circles(rng, n, r_lo, r_hi, lo, hi):
    r = rng.uniform(r_lo, r_hi, size=n)
    c = rng.uniform(lo, hi, size=(n, 2))
    return _f32(np.concatenate([c, r[:, None]], axis=1))


def ellipse_arclength_points(a, b, n, n_quad=400_000):
    """Points at arc lengths (i+1/2) P/n along the ellipse, with outward unit normals (G24)."""
    th = np.linspace(0.0, 2.0 * math.pi, n_quad + 1)
    x, y = a * np.cos(th), b * np.sin(th)
    seg = np.hypot(np.diff(x), np.diff(y))
    s = np.concatenate([[0.0], np.cumsum(seg)])
    P = s[-1]
    targets = (np.arange(n) + 0.5) * P / n
    th_i = np.interp(targets, s, th)
    px, py = a * np.cos(th_i), b * np.sin(th_i)
    nxv, nyv = px / (a * a), py / (b * b)
    nrm = np.hypot(nxv, nyv)
    return px, py, nxv / nrm, nyv / nrm, P


def track_circles(rng, a, b, n, r_lo, r_hi, off):
    px, py, nxv, nyv, _ = ellipse_arclength_points(a, b, n)
    o = rng.uniform(-off, off, size=n)
    r = rng.uniform(r_lo, r_hi, size=n)
    return _f32(np.stack([px + o * nxv, py + o * nyv, r], axis=1))


def rectangle_costmap(rng, n=512, res=0.05, n_rect=200, side_lo=0.2, side_hi=1.5):
    """Occupancy of the union of random axis-aligned rectangles, 5x5 box blur, zero padding (G26)."""
    size = n * res
    cx = rng.uniform(0.0, size, size=n_rect)
    cy = rng.uniform(0.0, size, size=n_rect)
    sx = rng.uniform(side_lo, side_hi, size=n_rect)
    sy = rng.uniform(side_lo, side_hi, size=n_rect)
    centres = (np.arange(n) + 0.5) * res
    occ = np.zeros((n, n), dtype=np.float64)  # [iy][ix]
    for i in range(n_rect):
        inx = np.abs(centres - cx[i]) <= 0.5 * sx[i]
        iny = np.abs(centres - cy[i]) <= 0.5 * sy[i]
        occ[np.ix_(iny, inx)] = 1.0
    pad = np.pad(occ, 2)
    blur = np.zeros_like(occ)
    for dy in range(5):
        for dx in range(5):
            blur += pad[dy:dy + n, dx:dx + n]
    return _f32(blur / 25.0)


# --------------------------------------------------------------------------- configs
_BICYCLE = dict(dyn=DYN_BICYCLE, dyn_p=[0.33], u_min=[-0.35, -3.0], u_max=[0.35, 3.0],
                sigma_eps=[0.1, 0.5], sigma_w=[0.02, 0.02, 0.01, 0.05])
_TRACK_NOM = [10.0, 6.0, 1.0, 5.0, 2.0, 4.0, 1000.0, 1.0]


def config0(K=256, M=16, T=20, near_obstacle=False) -> Problem:
    rng = np.random.default_rng(0)
    circles = random_circles(rng, 8, 0.3, 0.6, 0.0, 20.0)
    x0 = _f32([1.0, 1.0, 0.785, 2.0])
    if near_obstacle:  # supplementary scene: one obstacle 1.5 m ahead so the risk path is exercised
        circles = circles.copy()
        circles[0] = _f32([1.0 + 1.5 * math.cos(0.785), 1.0 + 1.5 * math.sin(0.785) + 0.25, 0.4])
    return Problem(name="C0" + ("-near" if near_obstacle else ""), K=K, M=M, T=T, dt=0.05, **_BICYCLE,
                   alpha=0.9, lam=1.0, gamma=1.0, nominal=NOM_GOAL, nom_p=[1.0, 18.0, 18.0, 1.0],
                   risk=RISK_CIRCLES, risk_p=[1000.0, 0.2], seed=0, x0=x0,
                   v=np.zeros((T, 2)), circles=circles)


def config1(K=2048, M=64, T=40, n_obs=32, seed=1) -> Problem:
    rng = np.random.default_rng(seed)
    circles = track_circles(rng, 10.0, 6.0, n_obs, 0.2, 0.4, 0.8)
    return Problem(name="C1", K=K, M=M, T=T, dt=0.05, **_BICYCLE, alpha=0.95, lam=0.5, gamma=0.5,
                   nominal=NOM_ELLIPSE_TRACK, nom_p=list(_TRACK_NOM), risk=RISK_CIRCLES,
                   risk_p=[1000.0, 0.2], seed=seed, x0=_f32([10.0, 0.0, math.pi / 2, 3.0]),
                   v=np.zeros((T, 2)), circles=circles)


def config2(K=8192, M=128, T=60) -> Problem:
    rng = np.random.default_rng(2)
    circles = track_circles(rng, 10.0, 6.0, 128, 0.2, 0.4, 0.8)
    return Problem(name="C2", K=K, M=M, T=T, dt=0.02, dyn=DYN_SINGLE_TRACK,
                   dyn_p=[4.0, 0.05, 0.17, 0.17, 30.0, 30.0, 0.5], u_min=[-0.35, -10.0],
                   u_max=[0.35, 10.0], sigma_eps=[0.1, 2.0],
                   sigma_w=[0.01, 0.01, 0.005, 0.05, 0.05, 0.05], alpha=0.95, lam=0.5, gamma=0.5,
                   nominal=NOM_ELLIPSE_TRACK, nom_p=list(_TRACK_NOM), risk=RISK_CIRCLES,
                   risk_p=[1000.0, 0.2], seed=2, x0=_f32([10.0, 0.0, math.pi / 2, 3.0, 0.0, 0.0]),
                   v=np.zeros((T, 2)), circles=circles)


def config3(K=16384, M=128, T=50) -> Problem:
    rng = np.random.default_rng(3)
    cmap = rectangle_costmap(rng)
    return Problem(name="C3", K=K, M=M, T=T, dt=0.05, **_BICYCLE, alpha=0.9, lam=1.0, gamma=1.0,
                   nominal=NOM_GOAL, nom_p=[1.0, 25.6, 25.6, 1.0], risk=RISK_COSTMAP,
                   risk_p=[1000.0], seed=3, x0=_f32([1.0, 1.0, 0.785, 2.0]), v=np.zeros((T, 2)),
                   costmap=cmap, map_res=0.05, map_ox=0.0, map_oy=0.0)


def config4(K=8192, M=64, T=50) -> Problem:
    """Config-1 track with 64 obstacles; sweep points and the closed loop vary K, M."""
    p = config1(K=K, M=M, T=T, n_obs=64, seed=4)
    return p.replace(name=f"C4-K{K}-M{M}")


def rounded_rect_points(ax, ay, rc, s_values):
    """Centreline points and outward unit normals of the rounded-rectangle track at arc lengths s
    (counter-clockwise from (ax+rc, 0)).  Scene geometry only (obstacle placement, start pose)."""
    seg = [2 * ay, rc * math.pi / 2, 2 * ax, rc * math.pi / 2] * 2          # straight, corner, ... from (ax+rc, -ay)
    P = sum(seg)
    pts = []
    for s in np.atleast_1d(s_values):
        u = (s + ay) % P                                                     # shift origin to the corner (ax+rc, -ay)
        corners = [(ax, ay), (-ax, ay), (-ax, -ay), (ax, -ay)]
        k = 0
        while u > seg[k]:
            u -= seg[k]; k += 1
        side, is_corner = k // 2, k % 2 == 1
        a0 = side * math.pi / 2                                              # outward normal angle of this side
        if not is_corner:
            n = (math.cos(a0), math.sin(a0)); t = (-math.sin(a0), math.cos(a0))
            start = [(ax + rc, -ay), (ax, ay + rc), (-ax - rc, ay), (-ax, -ay - rc)][side]
            pts.append((start[0] + u * t[0], start[1] + u * t[1], n[0], n[1]))
        else:
            c = corners[side]; ang = a0 + u / rc
            pts.append((c[0] + rc * math.cos(ang), c[1] + rc * math.sin(ang), math.cos(ang), math.sin(ang)))
    return np.array(pts), P


def paper_racing(K=1024, M=300, T=30, seed=5, single_track=False) -> Problem:
    """The paper's own controller set-up: costs (20)-(23) with c1..c5 = 2, 1, 0.1, 0.6, 2,
    l = q, horizon 30, lambda 0.35, eta 0.2, A 10, 1024 samples x 300 realisations, on a synthetic
    rounded-rectangle track with the published dimensions (0.6 m wide, 10.9 m centreline, 0.3 m corners, ten
    r = 0.1 m obstacles) because the paper's layout figure is missing.  Vehicle: kinematic bicycle
    at 1/28 scale (the paper's own model is not given)."""
    rc, hw = 0.3, 0.3
    ax = 1.5
    ay = (10.9 - 2 * math.pi * rc) / 4 - ax
    rng = np.random.default_rng(seed)
    P = 4 * (ax + ay) + 2 * math.pi * rc
    s_obs = (np.arange(10) + rng.uniform(0.2, 0.8, size=10)) * P / 10
    pts, _ = rounded_rect_points(ax, ay, rc, s_obs)
    off = rng.uniform(-0.18, 0.18, size=10)
    circles = _f32(np.stack([pts[:, 0] + off * pts[:, 2], pts[:, 1] + off * pts[:, 3], np.full(10, 0.1)], axis=1))
    start, _ = rounded_rect_points(ax, ay, rc, [P - ay - rc * math.pi / 2 - 0.6 * ax])   # on the bottom straight
    x0 = _f32([start[0, 0], start[0, 1], 0.0, 1.5])                                      # heading +x (counter-clockwise)
    if single_track:   # "dynamic vehicle model with tire dynamics", 1/28-scale linear-tyre stand-in
        veh = dict(dyn=DYN_SINGLE_TRACK, dyn_p=[0.15, 2.5e-4, 0.045, 0.045, 2.0, 2.0, 0.2], u_min=[-0.4, -0.6],
                   u_max=[0.4, 0.6], sigma_eps=[0.15, 0.15], sigma_w=[0.004, 0.004, 0.01, 0.03, 0.03, 0.1])
        x0 = _f32([start[0, 0], start[0, 1], 0.0, 1.5, 0.0, 0.0])
    else:
        veh = dict(dyn=DYN_BICYCLE, dyn_p=[0.093], u_min=[-0.4, -4.0], u_max=[0.4, 4.0], sigma_eps=[0.15, 1.0],
                   sigma_w=[0.004, 0.004, 0.01, 0.03])
    return Problem(name="paper-racing" + ("-st" if single_track else ""), K=K, M=M, T=T, dt=0.02, **veh, alpha=0.9, lam=0.35, gamma=0.35, A=10.0, B=1.0, C_u=0.5,
                   eta=0.2, nominal=NOM_RACING, nom_p=[ax, float(_f32(ay)), rc, hw, 2.0, 1.0, 0.1, 0.6, 2.0],
                   risk=RISK_NOMINAL, risk_p=[0.0], seed=seed, x0=x0, v=np.zeros((T, 2)), circles=circles)


C4_SWEEP_K = (1024, 4096, 16384, 65536)
C4_SWEEP_M = (16, 64, 256)


def small(p: Problem, K: int, M: Optional[int] = None, T: Optional[int] = None) -> Problem:
    """Same scene and parameters at a size the oracle finishes in seconds."""
    M = p.M if M is None else M
    T = p.T if T is None else T
    return p.replace(K=K, M=M, T=T, v=np.zeros((T, 2)) if T != p.T else p.v, name=f"{p.name}-K{K}")


def random_mean_control(p: Problem, seed: int, scale=(0.1, 0.5)) -> np.ndarray:
    """A non-zero mean control sequence (smooth random walk) so v-dependent terms are exercised."""
    rng = np.random.default_rng(1000 + seed)
    v = np.cumsum(rng.normal(size=(p.T, 2)), axis=0) / math.sqrt(p.T)
    return _f32(v * np.asarray(scale))


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}
