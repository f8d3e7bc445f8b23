"""Shared helpers of the GPU-vs-oracle parity tests (tolerances of BASELINE.json north_star)."""
import numpy as np

TOL_STATE_ABS = 1e-3     # rollout states at t = T: m, rad, m/s
TOL_COST_REL = 1e-4      # CVaR and total costs
TOL_V_ABS = 1e-4         # updated mean control


def rel_err(a, b):
    """|a-b| / max(|b|, s), s = median nonzero magnitude of b (G28); exact zeros must match."""
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    nz = np.abs(b[b != 0])
    s = float(np.median(nz)) if nz.size else 1.0
    return np.abs(a - b) / np.maximum(np.abs(b), s)


def assert_costs_close(a, b, what, tol=TOL_COST_REL):
    e = rel_err(a, b)
    assert e.max() <= tol, f"{what}: max rel err {e.max():.3e} at {np.unravel_index(e.argmax(), e.shape)}"


def gpu_outputs(ctl, p, iteration=0, x0=None, v=None, **kw):
    import torch
    d_x0 = ctl.tensor(p.x0 if x0 is None else x0)
    d_v = ctl.tensor(p.v if v is None else v)
    g = ctl.rollout_costs(d_x0, d_v, iteration, **kw)
    torch.cuda.synchronize()
    return {k: (t.cpu().numpy() if t is not None else None) for k, t in g.items()}


def check_rollout_parity(p, ctl, orc, iteration=0, x0=None, v=None, k_begin=0, k_end=None):
    """Stage-wise parity of A1-A7 (SURVEY.md section 8(c) 'How parity is checked')."""
    from oracle import oracle as O
    g = gpu_outputs(ctl, p, iteration, x0, v)
    r = orc.rollout_costs(x0=x0, v=v, iteration=iteration, k_begin=k_begin, k_end=k_end, n_threads=8)
    sl = slice(k_begin, k_end)
    gs = {k: a[sl] for k, a in g.items()}
    # A1: sampled controls
    assert np.abs(gs["u"] - r["u"]).max() < 2e-6 * max(1.0, np.abs(r["u"]).max()), "u"
    # A3: states at t = T
    ex = np.abs(gs["xT"] - r["xT"]).max()
    assert ex < TOL_STATE_ABS, f"xT abs err {ex:.3e}"
    # A2/A4: costs
    assert_costs_close(gs["S"], r["S"], "S")
    assert_costs_close(gs["L"], r["L"], "L")
    assert np.array_equal(gs["L"][r["L"] == 0] == 0, np.ones((r["L"] == 0).sum(), bool)) or \
        (gs["L"][r["L"] == 0] < 1e-4 * max(1.0, np.median(np.abs(r["L"][r["L"] != 0])) if (r["L"] != 0).any() else 1)).all()
    # A5/A6 isolated: the oracle's sort-based CVaR of the GPU's own L must equal the GPU's CVaR
    k_tail = O.tail_count(p.alpha, p.M)
    iso = np.array([O.cvar_topk(O.sensitivity_scale(gs["L"][i].astype(np.float64), p.B), k_tail)
                    for i in range(gs["L"].shape[0])])
    assert_costs_close(gs["cvar"], iso, "CVaR(select kernel) vs sort of GPU L", tol=2e-6)
    # end to end
    assert_costs_close(gs["cvar"], r["cvar"], "CVaR")
    assert_costs_close(gs["S_tilde"], r["S_tilde"], "S_tilde")
    return g, r


def check_update_parity(p, ctl, orc, r):
    """A8-A9 isolated: oracle S~ and u through the GPU weights/update kernel."""
    import torch
    d_S = ctl.tensor(r["S_tilde"].astype(np.float32))
    d_u = ctl.tensor(r["u"].astype(np.float32))
    g = ctl.weights_update(d_S, d_u)
    torch.cuda.synchronize()
    ref = orc.weights_update(r["S_tilde"].astype(np.float32).astype(np.float64),
                             r["u"].astype(np.float32).astype(np.float64))
    ev = np.abs(g["v_plus"].cpu().numpy() - ref["v_plus"]).max()
    assert ev < TOL_V_ABS, f"v+ (isolated update) abs err {ev:.3e}"
    w = g["w"].cpu().numpy()
    assert abs(w.sum() - 1.0) < 1e-5
    assert np.abs(w - ref["w"] / ref["Z"]).max() < 1e-5
    st = g["stats"].cpu().numpy()
    assert st[0] == np.float32(ref["beta"]) and abs(st[1] - ref["Z"]) < 1e-4 * ref["Z"]
    assert int(w.argmax()) == int(np.argmax(ref["w"])) or np.sort(ref["w"])[-2] > 1 - 1e-3


def check_step_parity(p, ctl, orc, r, iteration=0, x0=None, v=None):
    """End-to-end v+ (gap-aware: the softmin is one-hot at the BASELINE cost scales)."""
    import torch
    d_x0 = ctl.tensor(p.x0 if x0 is None else x0)
    d_v = ctl.tensor(p.v if v is None else v)
    ctl.step(d_x0, d_v, iteration)
    torch.cuda.synchronize()
    vp = d_v.cpu().numpy()
    ref = orc.weights_update(r["S_tilde"], r["u"])
    err = np.abs(vp - ref["v_plus"]).max()
    if err < TOL_V_ABS:
        return "match", err
    # The softmin is sharp at the BASELINE cost scales: fp32 error in q perturbs the weights by
    # exp(+-dS/lambda).  Isolate A8-A9: the GPU's own fp64 S~ through the oracle's update must
    # reproduce the GPU's v+.
    _, St = ctl.costs_f64()
    St = St.cpu().numpy()
    ref2 = orc.weights_update(St, r["u"])
    err2 = np.abs(vp - ref2["v_plus"]).max()
    assert err2 < TOL_V_ABS, f"v+ with GPU S~ through oracle update: {err2:.3e}"
    dS = np.abs(St - r["S_tilde"])
    return f"weight-sensitive (end-to-end err {err:.2e}, max|dS~| {dS.max():.2e}, lambda {p.lam})", err
