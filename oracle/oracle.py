"""ctypes front end of the fp64 C++ oracle (TEST INFRASTRUCTURE, not the product).

Takes any object with the attributes of ``workloads.Problem`` (duck-typed: this
module imports neither the workloads module nor the CUDA package).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class OrcProblem(C.Structure):
    _fields_ = [
        ("K", C.c_int32), ("M", C.c_int32), ("T", C.c_int32),
        ("dt", C.c_double),
        ("dyn", C.c_int32), ("dyn_p", C.c_double * 8),
        ("u_min", C.c_double * 2), ("u_max", C.c_double * 2),
        ("sigma_eps", C.c_double * 2), ("sigma_w", C.c_double * 6),
        ("alpha", C.c_double), ("lam", C.c_double), ("gamma", C.c_double),
        ("A", C.c_double), ("B", C.c_double), ("C_u", C.c_double), ("eta", C.c_double),
        ("nominal", C.c_int32), ("nom_p", C.c_double * 12),
        ("risk", C.c_int32), ("risk_p", C.c_double * 4),
        ("noise_kind", C.c_int32), ("noise_p", C.c_double * 4),
        ("seed", C.c_uint64),
        ("circles", C.POINTER(C.c_double)), ("n_circles", C.c_int32),
        ("costmap", C.POINTER(C.c_double)), ("map_h", C.c_int32), ("map_w", C.c_int32),
        ("map_res", C.c_double), ("map_ox", C.c_double), ("map_oy", C.c_double),
    ]


_DP = C.POINTER(C.c_double)
_U32P = C.POINTER(C.c_uint32)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_philox4x32_10.argtypes = [_U32P, _U32P, _U32P]
        L.orc_counter.argtypes = [C.c_uint32] * 6 + [C.c_uint64, _U32P]
        L.orc_box_muller.argtypes = [C.c_uint32, C.c_uint32, _DP]
        L.orc_box_muller16.argtypes = [C.c_uint32, _DP]
        L.orc_state_noise.argtypes = [C.POINTER(OrcProblem), C.c_uint32, C.c_uint32, C.c_uint32,
                                      C.c_uint32, C.c_uint64, _DP]
        L.orc_nx.argtypes = [C.c_int32]
        L.orc_dynamics.argtypes = [C.POINTER(OrcProblem), _DP, _DP, _DP]
        for f in (L.orc_q, L.orc_l):
            f.argtypes = [C.POINTER(OrcProblem), _DP]
            f.restype = C.c_double
        L.orc_phi.argtypes = [C.POINTER(OrcProblem), _DP, _DP]
        L.orc_phi.restype = C.c_double
        for f in (L.orc_racing_offset, L.orc_racing_arclength, L.orc_indicator_margin, L.orc_hinge_margin):
            f.argtypes = [C.POINTER(OrcProblem), C.c_double, C.c_double]
            f.restype = C.c_double
        L.orc_ellipse_offset.argtypes = [C.c_double] * 4
        L.orc_ellipse_offset.restype = C.c_double
        L.orc_bilinear.argtypes = [C.POINTER(OrcProblem), C.c_double, C.c_double]
        L.orc_bilinear.restype = C.c_double
        L.orc_tail_count.argtypes = [C.c_double, C.c_int32]
        L.orc_tail_count.restype = C.c_int32
        L.orc_cvar_topk.argtypes = [_DP, C.c_int32, C.c_int32]
        L.orc_cvar_topk.restype = C.c_double
        L.orc_cvar_literal12.argtypes = [_DP, C.c_int32, C.c_double]
        L.orc_cvar_literal12.restype = C.c_double
        L.orc_sensitivity_scale.argtypes = [_DP, C.c_int32, C.c_double, _DP]
        L.orc_rollout_costs.argtypes = [C.POINTER(OrcProblem), _DP, _DP, C.c_uint64, C.c_int32,
                                        C.c_int32, C.c_int32] + [_DP] * 8
        L.orc_rollout_costs.restype = C.c_int
        L.orc_weights_update.argtypes = [C.POINTER(OrcProblem), _DP, _DP, _DP, _DP, _DP, _DP]
        L.orc_weights_update.restype = C.c_int
        L.orc_step.argtypes = [C.POINTER(OrcProblem), _DP, _DP, C.c_uint64, C.c_int32, _DP]
        L.orc_step.restype = C.c_int
        L.orc_plant_step.argtypes = [C.POINTER(OrcProblem), _DP, _DP, C.c_uint64, _DP]
        L.orc_shift.argtypes = [_DP, C.c_int32, _DP]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(_DP) if a is not None else None


def _vec(dst, src):
    src = list(src)
    for i in range(len(dst)):
        dst[i] = float(src[i]) if i < len(src) else 0.0


class Oracle:
    """The oracle bound to one problem (keeps the environment arrays alive)."""

    def __init__(self, p):
        lib()
        self.p = p
        s = OrcProblem()
        s.K, s.M, s.T, s.dt = int(p.K), int(p.M), int(p.T), float(p.dt)
        s.dyn, s.nominal, s.risk = int(p.dyn), int(p.nominal), int(p.risk)
        _vec(s.dyn_p, p.dyn_p); _vec(s.u_min, p.u_min); _vec(s.u_max, p.u_max)
        _vec(s.sigma_eps, p.sigma_eps); _vec(s.sigma_w, p.sigma_w)
        s.alpha, s.lam, s.gamma = float(p.alpha), float(p.lam), float(p.gamma)
        s.A, s.B, s.C_u, s.eta = float(p.A), float(p.B), float(p.C_u), float(p.eta)
        _vec(s.nom_p, p.nom_p); _vec(s.risk_p, p.risk_p)
        s.noise_kind = int(getattr(p, "noise_kind", 0))
        _vec(s.noise_p, getattr(p, "noise_p", [0, 0, 0, 0]))
        s.seed = int(p.seed)
        self._circles = self._costmap = None
        if getattr(p, "circles", None) is not None:
            self._circles = np.ascontiguousarray(p.circles, dtype=np.float64)
            s.circles, s.n_circles = _dp(self._circles), int(self._circles.shape[0])
        if getattr(p, "costmap", None) is not None:
            self._costmap = np.ascontiguousarray(p.costmap, dtype=np.float64)
            s.costmap = _dp(self._costmap)
            s.map_h, s.map_w = int(self._costmap.shape[0]), int(self._costmap.shape[1])
            s.map_res, s.map_ox, s.map_oy = float(p.map_res), float(p.map_ox), float(p.map_oy)
        self.s = s
        self.nx = lib().orc_nx(s.dyn)

    # ---- models
    def dynamics(self, x, u):
        x = np.ascontiguousarray(x, dtype=np.float64); u = np.ascontiguousarray(u, dtype=np.float64)
        out = np.zeros(self.nx)
        lib().orc_dynamics(C.byref(self.s), _dp(x), _dp(u), _dp(out))
        return out

    def q(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        return lib().orc_q(C.byref(self.s), _dp(x))

    def phi(self, x, x0=None):
        x = np.ascontiguousarray(x, dtype=np.float64)
        x0 = np.ascontiguousarray(self.p.x0 if x0 is None else x0, dtype=np.float64)
        return lib().orc_phi(C.byref(self.s), _dp(x), _dp(x0))

    def racing_offset(self, X, Y):
        return lib().orc_racing_offset(C.byref(self.s), float(X), float(Y))

    def racing_arclength(self, X, Y):
        return lib().orc_racing_arclength(C.byref(self.s), float(X), float(Y))

    def indicator_margin(self, X, Y):
        return lib().orc_indicator_margin(C.byref(self.s), float(X), float(Y))

    def hinge_margin(self, X, Y):
        return lib().orc_hinge_margin(C.byref(self.s), float(X), float(Y))

    def l(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        return lib().orc_l(C.byref(self.s), _dp(x))

    def bilinear(self, X, Y):
        return lib().orc_bilinear(C.byref(self.s), float(X), float(Y))

    def state_noise(self, k, m, t, stream, iteration):
        w = np.zeros(6)
        lib().orc_state_noise(C.byref(self.s), k, m, t, stream, iteration, _dp(w))
        return w[: self.nx]

    # ---- iteration
    def rollout_costs(self, x0=None, v=None, iteration=0, k_begin=0, k_end=None, n_threads=1,
                      want_L=True, want_xT=True, want_margin=False):
        p, s = self.p, self.s
        x0 = np.ascontiguousarray(p.x0 if x0 is None else x0, dtype=np.float64)
        v = np.ascontiguousarray(p.v if v is None else v, dtype=np.float64)
        k_end = s.K if k_end is None else k_end
        n = k_end - k_begin
        out = dict(
            u=np.zeros((n, s.T, 2)), S=np.zeros(n), cvar=np.zeros(n), S_tilde=np.zeros(n),
            L=np.zeros((n, s.M)) if want_L else None,
            xT=np.zeros((n, s.M, self.nx)) if want_xT else None,
            x_nom=np.zeros((n, self.nx)),
            margin=np.zeros((n, s.M + 1)) if want_margin else None,
        )
        rc = lib().orc_rollout_costs(C.byref(s), _dp(x0), _dp(v), int(iteration), k_begin, k_end,
                                     int(n_threads), _dp(out["u"]), _dp(out["S"]), _dp(out["cvar"]),
                                     _dp(out["S_tilde"]), _dp(out["L"]), _dp(out["xT"]),
                                     _dp(out["x_nom"]), _dp(out["margin"]))
        if rc:
            raise RuntimeError(f"orc_rollout_costs failed: {rc}")
        return out

    def weights_update(self, S_tilde, u):
        s = self.s
        S_tilde = np.ascontiguousarray(S_tilde, dtype=np.float64)
        u = np.ascontiguousarray(u, dtype=np.float64)
        assert S_tilde.shape == (s.K,) and u.shape == (s.K, s.T, 2)
        vp, w = np.zeros((s.T, 2)), np.zeros(s.K)
        Z, beta = C.c_double(), C.c_double()
        lib().orc_weights_update(C.byref(s), _dp(S_tilde), _dp(u), _dp(vp), _dp(w),
                                 C.cast(C.byref(Z), _DP), C.cast(C.byref(beta), _DP))
        return dict(v_plus=vp, w=w, Z=Z.value, beta=beta.value)

    def step(self, x0=None, v=None, iteration=0, n_threads=1):
        p, s = self.p, self.s
        x0 = np.ascontiguousarray(p.x0 if x0 is None else x0, dtype=np.float64)
        v = np.ascontiguousarray(p.v if v is None else v, dtype=np.float64)
        vp = np.zeros((s.T, 2))
        rc = lib().orc_step(C.byref(s), _dp(x0), _dp(v), int(iteration), int(n_threads), _dp(vp))
        if rc:
            raise RuntimeError(f"orc_step failed: {rc}")
        return vp

    def plant_step(self, x0, u0, iteration):
        x0 = np.ascontiguousarray(x0, dtype=np.float64); u0 = np.ascontiguousarray(u0, dtype=np.float64)
        out = np.zeros(self.nx)
        lib().orc_plant_step(C.byref(self.s), _dp(x0), _dp(u0), int(iteration), _dp(out))
        return out


# ---- free functions
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def counter(k, m, t, J, j, stream, iteration):
    o = (C.c_uint32 * 4)()
    lib().orc_counter(k, m, t, J, j, stream, iteration, o)
    return [int(x) for x in o]


def box_muller(ra, rb):
    z = np.zeros(2)
    lib().orc_box_muller(int(ra), int(rb), _dp(z))
    return z


def box_muller16(w):
    z = np.zeros(2)
    lib().orc_box_muller16(int(w), _dp(z))
    return z


def tail_count(alpha, M):
    return lib().orc_tail_count(float(alpha), int(M))


def cvar_topk(L, k_tail):
    L = np.ascontiguousarray(L, dtype=np.float64)
    return lib().orc_cvar_topk(_dp(L), L.size, int(k_tail))


def cvar_literal12(L, alpha):
    L = np.ascontiguousarray(L, dtype=np.float64)
    return lib().orc_cvar_literal12(_dp(L), L.size, float(alpha))


def sensitivity_scale(L, B):
    L = np.ascontiguousarray(L, dtype=np.float64)
    out = np.zeros_like(L)
    lib().orc_sensitivity_scale(_dp(L), L.size, float(B), _dp(out))
    return out


def ellipse_offset(a, b, X, Y):
    return lib().orc_ellipse_offset(float(a), float(b), float(X), float(Y))


def shift(v_plus):
    v_plus = np.ascontiguousarray(v_plus, dtype=np.float64)
    out = np.zeros_like(v_plus)
    lib().orc_shift(_dp(v_plus), v_plus.shape[0], _dp(out))
    return out


def host_cores():
    return os.cpu_count() or 1


# ---- K-sharded update (not in the paper): (17) PAPER.md:134 and (4) :51 written per shard.
# Factor exp(-(beta_g - beta)/lambda) out of every weight of shard g: sum_k w_k u_k = sum_g s_g N_g, Z = sum_g s_g Z_g.
def shard_partial(S_tilde, u, lam):
    """{beta_g, Z_g, N_g[T,2]} (flat [2+2T]) of the samples of one shard: S_tilde [K_g], u [K_g,T,2]."""
    S_tilde = np.asarray(S_tilde, dtype=np.float64)
    u = np.asarray(u, dtype=np.float64)
    beta = S_tilde.min()
    w = np.exp(-(S_tilde - beta) / lam)
    N = np.zeros(u.shape[1:])
    for k in range(u.shape[0]):
        N += w[k] * u[k]
    return np.concatenate([[beta, w.sum()], N.ravel()])


def combine_partials(parts, lam, u_min, u_max):
    """v+ [T,2] from the shards' partials [G, 2+2T] (any order)."""
    parts = np.asarray(parts, dtype=np.float64)
    beta = parts[:, 0].min()
    s = np.exp(-(parts[:, 0] - beta) / lam)
    Z = float((s * parts[:, 1]).sum())
    N = (s[:, None] * parts[:, 2:]).sum(axis=0).reshape(-1, 2)
    return np.clip(N / Z, np.asarray(u_min, dtype=np.float64), np.asarray(u_max, dtype=np.float64))
