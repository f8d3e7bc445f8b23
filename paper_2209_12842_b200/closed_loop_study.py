"""Closed-loop RA-MPPI vs baseline MPPI on the synthetic race track.

    python -m paper_2209_12842_b200.closed_loop_study [--iterations 3000] [--noise gaussian|uniform|jump]

Runs the receding-horizon loop (CUDA graph, simulated plant) twice on the paper's own controller set-up
(costs (20)-(23)): RA-MPPI with 1024 samples x 300 realisations and A = 10, and the baseline
MPPI (A = 0) with the same total number of sampled trajectories (last sentence), then counts
collisions the way PAPER.md:263 defines them (the state is inside an obstacle or outside the track) and laps.
All control computation runs in libra_mppi.so; this module only post-processes the logged states
(lap / collision bookkeeping is outside the hot path).  The track is the synthetic stand-in of workloads.py, so
the numbers are not the paper's (its track layout, vehicle model and C_u are unpublished).  On this benign
stand-in both controllers collide about once per 3000 iterations, so it does not separate their collision rates;
what it does show is the price of the risk term: with the paper's A = 10 the RA-MPPI controller drives far more
slowly until C_u is raised towards the typical CVaR (--C_u 8: lap time 6.6 s against the baseline's 4.1 s).
"""
from __future__ import annotations

import argparse
import json
import math

import numpy as np

from . import workloads as W


def track_metrics(p, log):
    """Collision events, laps and lap time from the closed-loop log (states after each plant step)."""
    ax, ay, rc, hw = p.nom_p[:4]
    X, Y = log[:, 0].astype(np.float64), log[:, 1].astype(np.float64)
    qx, qy = np.abs(X) - ax, np.abs(Y) - ay
    sd = np.hypot(np.maximum(qx, 0), np.maximum(qy, 0)) + np.minimum(np.maximum(qx, qy), 0)
    off_track = np.abs(sd - rc) > hw
    c = np.asarray(p.circles, dtype=np.float64)
    in_obstacle = (np.hypot(X[:, None] - c[None, :, 0], Y[:, None] - c[None, :, 1]) < c[None, :, 2]).any(axis=1)
    bad = off_track | in_obstacle
    events = int(np.count_nonzero(bad[1:] & ~bad[:-1]) + int(bad[0]))
    ang = np.unwrap(np.arctan2(Y, X))
    laps = float((ang[-1] - ang[0]) / (2 * math.pi))
    return {"collision_events": events, "steps_in_collision": int(bad.sum()), "off_track_steps": int(off_track.sum()),
            "obstacle_steps": int(in_obstacle.sum()), "laps": laps,
            "collisions_per_lap": events / laps if laps > 0.05 else None,
            "lap_time_s": len(log) * p.dt / laps if laps > 0.05 else None,
            "mean_speed": float(log[:, 3].mean())}


def run(p, iterations, device=0):
    import torch

    from .controller import RaMppi
    ctl = RaMppi(p, device=device)
    d_x0, d_v = ctl.tensor(p.x0), ctl.tensor(np.zeros((p.T, 2)))
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(torch.cuda.current_stream())
    log, _ = ctl.closed_loop(d_x0, d_v, 0, iterations, log=True, timing=False)
    b.record(torch.cuda.current_stream())
    b.synchronize()
    out = track_metrics(p, log.cpu().numpy())
    out["controller_hz"] = iterations / (a.elapsed_time(b) * 1e-3)
    ctl.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--iterations", type=int, default=3000)
    ap.add_argument("--noise", default="gaussian", choices=["gaussian", "uniform", "jump"])
    ap.add_argument("--alpha", type=float, default=0.9)
    ap.add_argument("--C_u", type=float, default=0.5)
    args = ap.parse_args()
    base = W.paper_racing()
    if args.noise == "uniform":      # uniform disturbance
        base = base.replace(noise_kind=W.NOISE_UNIFORM, sigma_w=[s * math.sqrt(3.0) for s in base.sigma_w])
    elif args.noise == "jump":       # 2 % chance of a sudden change in an arbitrary direction
        base = base.replace(noise_kind=W.NOISE_JUMP, noise_p=[0.02, 0, 0, 0], sigma_w=[s * 7.0 for s in base.sigma_w])
    ra = base.replace(alpha=args.alpha, C_u=args.C_u)
    mppi = base.replace(A=0.0, K=base.K * base.M, M=1, name="paper-racing-MPPI")   # same number of trajectories
    for name, p in (("RA-MPPI", ra), ("MPPI", mppi)):
        r = run(p, args.iterations)
        print(json.dumps({"controller": name, "noise": args.noise, "K": p.K, "M": p.M, "A": p.A, "alpha": p.alpha,
                          "C_u": p.C_u, "iterations": args.iterations, **r}), flush=True)


if __name__ == "__main__":
    main()
