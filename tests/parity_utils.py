"""Shared helpers of the GPU-vs-oracle parity tests (tolerances of BASELINE.json north_star)."""
import numpy as np

TOL_STATE_ABS = 1e-3     # rollout states at t = T: m, rad, m/s
TOL_COST_REL = 1e-4      # CVaR and total costs
TOL_V_ABS = 1e-4         # updated mean control
ZERO_MARGIN_M = 1e-5     # "exact zeros must match" (G28) away from an obstacle rim by more than this
ZERO_LEAK_REL = 1e-4     # risk kinds without a rim: GPU L where the oracle's is exactly 0, relative to the typical cost
BOUND_MAX = 10 * 1e-4    # a v+ fallback verdict whose weight-sensitivity bound exceeds 10 TOL_V_ABS proves too little: fail

# every end-to-end v+ comparison of the session: (case, verdict, err, max|dS~|, gap of the two smallest S~, bound);
# tests/conftest.py prints the tally and writes gpurun_out/parity_verdicts.md at session end
VERDICTS = []


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


def check_rollout_parity(p, ctl, orc, iteration=0, x0=None, v=None, k_begin=0, k_end=None, tol_cost=TOL_COST_REL):
    """Stage-wise parity of A1-A7 (SURVEY.md section 8(c) 'How parity is checked').  tol_cost is north_star's 1e-4
    everywhere except the one stress case that documents where it stops holding (yaw winding, test_gpu_parity.py)."""
    from oracle import oracle as O
    g = gpu_outputs(ctl, p, iteration, x0, v)
    hinge = p.risk == 0          # circle risk: the oracle also reports each rollout's closest approach to a rim
    r = orc.rollout_costs(x0=x0, v=v, iteration=iteration, k_begin=k_begin, k_end=k_end, n_threads=8,
                          want_margin=hinge)
    sl = slice(k_begin, k_end)
    gs = {k: a[sl] for k, a in g.items()}
    # A1: sampled controls
    assert np.abs(gs["u"] - r["u"]).max() < 2e-6 * max(1.0, np.abs(r["u"]).max()), "u"
    # A3: states at t = T
    ex = np.abs(gs["xT"] - r["xT"]).max()
    assert ex < TOL_STATE_ABS, f"xT abs err {ex:.3e}"
    # A2/A4: costs
    assert_costs_close(gs["S"], r["S"], "S", tol=tol_cost)
    assert_costs_close(gs["L"], r["L"], "L", tol=tol_cost)
    if hinge:
        # exact zeros must match (G28): a rollout the oracle scores exactly 0 and whose closest approach to
        # any rim r + margin exceeds ZERO_MARGIN_M must be exactly 0 on the GPU too (exact culling, no leakage); within
        # ZERO_MARGIN_M of a rim both answers are correct and the relative tolerance above already bounds the value
        clear = (r["L"] == 0) & (r["margin"][:, 1:] > ZERO_MARGIN_M)
        assert (gs["L"][clear] == 0).all(), f"{(gs['L'][clear] != 0).sum()} rollouts clear of every obstacle have L != 0"
        # and the other way round: nothing the oracle scores > 0 clear of a rim may vanish on the GPU
        inside = (r["L"] > 0) & (r["margin"][:, 1:] > ZERO_MARGIN_M)
        assert (gs["L"][inside] > 0).all()
    else:
        # the other risk kinds (costmap, linear, l = q) have no rim diagnostic, but a rollout the oracle scores exactly 0
        # may still not pick up more than rounding on the GPU: a bilinear lookup one texel off, or a leaked term, is far
        # above ZERO_LEAK_REL of the typical cost (a position error of 1e-6 m across a cell edge of the BASELINE costmap
        # is worth about 1e-6 / res * weight = 0.02 against typical costs of 1e3 and more)
        zero = r["L"] == 0
        if zero.any():
            nz = np.abs(r["L"][r["L"] != 0])
            scale = float(np.median(nz)) if nz.size else 1.0
            leak = float(np.abs(gs["L"][zero]).max())
            assert leak <= ZERO_LEAK_REL * scale, (f"{int((gs['L'][zero] != 0).sum())} of {int(zero.sum())} rollouts the oracle "
                                                   f"scores 0 have L up to {leak:.3e} on the GPU (typical cost {scale:.3e})")
    # A5/A6 isolated: the oracle's sort-based CVaR of the GPU's own L must equal the GPU's CVaR
    k_tail = O.tail_count(p.alpha, p.M)
    iso = np.array([O.cvar_topk(O.sensitivity_scale(gs["L"][i].astype(np.float64), p.B), k_tail)
                    for i in range(gs["L"].shape[0])])
    assert_costs_close(gs["cvar"], iso, "CVaR(select kernel) vs sort of GPU L", tol=2e-6)
    # end to end
    assert_costs_close(gs["cvar"], r["cvar"], "CVaR", tol=tol_cost)
    assert_costs_close(gs["S_tilde"], r["S_tilde"], "S_tilde", tol=tol_cost)
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


def check_step_parity(p, ctl, orc, r, iteration=0, x0=None, v=None, case=None):
    """End-to-end v+ against the oracle.

    "match": |v+ - oracle v+| < 1e-4 outright.  Otherwise the mismatch must be explained, and bounded, by the
    sensitivity of the softmin (17) to the fp32 error dS~ of the costs -- the softmin is one-hot at the BASELINE cost
    scales, so two near-tied minima can swap:
      (a) A8-A9 in isolation: the GPU's own fp64 S~ through the ORACLE's update reproduces the GPU's v+ to 1e-4;
      (b) a rigorous bound: perturbing every S~_k by at most D changes each normalised weight by a factor within
          exp(+-2D/lambda), hence |dv+| <= (exp(2D/lambda) - 1) max_{t,i} sum_k w_k |u_k - v+| (clamping is 1-Lipschitz).
          D = max |dS~| over the samples that can carry weight (S~ - beta <= 30 lambda on either side); the rest hold at
          most K exp(-30) of the weight.  The observed error must lie within that bound.
    The verdict says which it was: "near-tie" when the two smallest oracle S~ are closer than 2D (SURVEY's condition),
    else "weight-sensitive".  Every call is recorded in VERDICTS."""
    import torch
    d_x0 = ctl.tensor(p.x0 if x0 is None else x0)
    d_v = ctl.tensor(p.v if v is None else v)
    ctl.step(d_x0, d_v, iteration)
    torch.cuda.synchronize()
    vp = d_v.cpu().numpy()
    ref = orc.weights_update(r["S_tilde"], r["u"])
    err = float(np.abs(vp - ref["v_plus"]).max())
    name = case or f"{p.name} K={p.K} M={p.M} T={p.T} lambda={p.lam:g}"
    s2 = np.sort(r["S_tilde"])[:2]
    gap = float(s2[1] - s2[0]) if s2.size > 1 else float("inf")
    if err < TOL_V_ABS:
        VERDICTS.append((name, "match", err, None, gap, None))
        return "match", err
    _, St = ctl.costs_f64()
    St = St.cpu().numpy()
    ref2 = orc.weights_update(St, r["u"])
    err2 = np.abs(vp - ref2["v_plus"]).max()
    assert err2 < TOL_V_ABS, f"v+ with GPU S~ through oracle update: {err2:.3e}"              # (a)
    live = ((r["S_tilde"] - r["S_tilde"].min()) <= 30 * p.lam) | ((St - St.min()) <= 30 * p.lam)
    D = float(np.abs(St - r["S_tilde"])[live].max())
    w = ref["w"] / ref["Z"]
    mad = np.einsum("k,kti->ti", w, np.abs(r["u"] - ref["v_plus"][None])).max()
    span = np.abs(r["u"] - ref["v_plus"][None]).max()
    bound = TOL_V_ABS + float(np.expm1(2 * D / p.lam)) * mad + p.K * np.exp(-30.0) * span
    assert err <= bound, f"v+ err {err:.3e} exceeds the weight-sensitivity bound {bound:.3e} (max|dS~| {D:.3e}, lambda {p.lam})"   # (b)
    # the bound is rigorous but loose at small lambda (D = 1e-2 at lambda = 0.5 admits 4 % of the spread): a verdict that
    # rests on a bound this wide could hide an update bug, so such a case must be re-posed (larger lambda, other seed)
    assert bound <= BOUND_MAX, (f"v+ err {err:.3e} is within its weight-sensitivity bound {bound:.3e}, but a bound above "
                                f"{BOUND_MAX:.0e} is too loose to count as parity (max|dS~| {D:.3e}, lambda {p.lam})")
    kind = "near-tie" if gap < 2 * D else "weight-sensitive"
    VERDICTS.append((name, kind, err, D, gap, bound))
    return f"{kind} (end-to-end err {err:.2e} <= bound {bound:.2e}; max|dS~| {D:.2e}, gap {gap:.2e}, lambda {p.lam})", err
