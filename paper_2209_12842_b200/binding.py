"""Thin ctypes binding of libra_mppi.so (argument marshalling only).

Function names mirror include/ra_mppi.h.  Every step of the path runs in the CUDA kernels
behind the C ABI; torch is used only for device buffers and streams.  There is no CPU
fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libra_mppi.so")

RA_OK, RA_EINVAL, RA_EUNSUPPORTED, RA_ECUDA, RA_ENOMEM = range(5)
_STATUS = {0: "RA_OK", 1: "RA_EINVAL", 2: "RA_EUNSUPPORTED", 3: "RA_ECUDA", 4: "RA_ENOMEM"}


class RaMppiError(RuntimeError):
    def __init__(self, status, where, detail=""):
        self.status = status
        super().__init__(f"{where}: {_STATUS.get(status, status)} {detail}".strip())


class ra_mppi_config(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32),
        ("K", C.c_int32), ("M", C.c_int32), ("T", C.c_int32),
        ("dt", C.c_float),
        ("dyn", C.c_int32), ("dyn_p", C.c_float * 8),
        ("u_min", C.c_float * 2), ("u_max", C.c_float * 2),
        ("sigma_eps", C.c_float * 2), ("sigma_w", C.c_float * 6),
        ("alpha", C.c_float), ("lam", C.c_float), ("gamma", C.c_float),
        ("A", C.c_float), ("B", C.c_float), ("C_u", C.c_float), ("eta", C.c_float),
        ("nominal", C.c_int32), ("nom_p", C.c_float * 12),
        ("risk", C.c_int32), ("risk_p", C.c_float * 4),
        ("noise_kind", C.c_int32), ("noise_p", C.c_float * 4),
        ("noise_mode", C.c_int32),
        ("seed", C.c_uint64),
        ("device", C.c_int32),
        ("k_offset", C.c_int32), ("K_total", C.c_int32),
    ]


class ra_mppi_env(C.Structure):
    _fields_ = [
        ("circles", C.POINTER(C.c_float)), ("n_circles", C.c_int32),
        ("costmap", C.POINTER(C.c_float)), ("map_h", C.c_int32), ("map_w", C.c_int32),
        ("map_res", C.c_float), ("map_ox", C.c_float), ("map_oy", C.c_float),
    ]


EXPORTS = (
    "ra_mppi_create", "ra_mppi_create_error", "ra_mppi_set_env", "ra_mppi_step", "ra_mppi_rollout_costs", "ra_mppi_weights_update",
    "ra_mppi_weights_update_static", "ra_mppi_weights_update_static_error",
    "ra_mppi_step_partial", "ra_mppi_combine_partials",
    "ra_mppi_step_host", "ra_mppi_enable_kernel_timing", "ra_mppi_last_rollout_ms",
    "ra_mppi_export_costs_f64", "ra_mppi_plant_shift", "ra_mppi_closed_loop", "ra_mppi_philox", "ra_mppi_state_noise",
    "ra_mppi_measure_pipe_peaks", "ra_mppi_query_counts", "ra_mppi_rollout_variant", "ra_mppi_launches_per_step", "ra_mppi_last_error", "ra_mppi_destroy",
)

_lib = None


def load():
    """Load libra_mppi.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        _lib = open_library(LIB_PATH)
    return _lib


def open_library(path):
    """A configured ctypes handle of the library at `path` (the product library, or the checked build the tests use)."""
    if not os.path.exists(path):
        raise RaMppiError(RA_ECUDA, "load",
                          f"{path} is missing: run `python -m paper_2209_12842_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(path)
    vp, fp, u64, i32 = C.c_void_p, C.c_void_p, C.c_uint64, C.c_int32
    L.ra_mppi_create.argtypes = [C.POINTER(ra_mppi_config), C.POINTER(ra_mppi_env), C.POINTER(vp)]
    L.ra_mppi_create_error.argtypes = []
    L.ra_mppi_create_error.restype = C.c_char_p
    L.ra_mppi_set_env.argtypes = [vp, C.POINTER(ra_mppi_env)]
    L.ra_mppi_step.argtypes = [vp, fp, fp, u64, vp]
    L.ra_mppi_rollout_costs.argtypes = [vp, fp, fp, u64, fp, fp, fp, fp, fp, fp, vp]
    L.ra_mppi_step_partial.argtypes = [vp, fp, fp, u64, vp, vp]
    L.ra_mppi_combine_partials.argtypes = [vp, vp, i32, fp, vp]
    L.ra_mppi_weights_update.argtypes = [vp, fp, fp, fp, fp, fp, vp]
    L.ra_mppi_weights_update_static.argtypes = [i32, i32, C.c_float, C.POINTER(C.c_float), C.POINTER(C.c_float),
                                                fp, fp, fp, vp]
    L.ra_mppi_weights_update_static_error.argtypes = []
    L.ra_mppi_weights_update_static_error.restype = C.c_char_p
    L.ra_mppi_export_costs_f64.argtypes = [vp, vp, vp, vp]
    L.ra_mppi_step_host.argtypes = [vp, vp, vp, u64, vp]
    L.ra_mppi_enable_kernel_timing.argtypes = [vp, i32]
    L.ra_mppi_last_rollout_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.ra_mppi_plant_shift.argtypes = [vp, fp, fp, fp, u64, vp]
    L.ra_mppi_closed_loop.argtypes = [vp, fp, fp, u64, i32, fp, C.POINTER(C.c_float), vp]
    L.ra_mppi_philox.argtypes = [vp, vp, i32, vp, vp]
    L.ra_mppi_state_noise.argtypes = [vp, vp, i32, u64, fp, vp]
    L.ra_mppi_measure_pipe_peaks.argtypes = [i32, C.POINTER(C.c_float)]
    L.ra_mppi_query_counts.argtypes = [C.POINTER(ra_mppi_config), C.POINTER(i32), C.POINTER(i32)]
    L.ra_mppi_rollout_variant.argtypes = [vp, C.POINTER(i32)]
    L.ra_mppi_launches_per_step.argtypes = [vp]
    L.ra_mppi_launches_per_step.restype = i32
    L.ra_mppi_last_error.argtypes = [vp]
    L.ra_mppi_last_error.restype = C.c_char_p
    L.ra_mppi_destroy.argtypes = [vp]
    for name in EXPORTS:
        if name not in ("ra_mppi_launches_per_step", "ra_mppi_last_error", "ra_mppi_weights_update_static_error", "ra_mppi_create_error"):
            getattr(L, name).restype = C.c_int
    return L


def _fill(dst, src):
    src = list(src)
    for i in range(len(dst)):
        dst[i] = float(src[i]) if i < len(src) else 0.0


def make_config(p, device=0) -> ra_mppi_config:
    """Marshal a workloads.Problem-like record into the C struct (fp32)."""
    c = ra_mppi_config()
    c.struct_size = C.sizeof(ra_mppi_config)
    c.K, c.M, c.T, c.dt = int(p.K), int(p.M), int(p.T), float(p.dt)
    c.dyn, c.nominal, c.risk = int(p.dyn), int(p.nominal), int(p.risk)
    _fill(c.dyn_p, p.dyn_p); _fill(c.u_min, p.u_min); _fill(c.u_max, p.u_max)
    _fill(c.sigma_eps, p.sigma_eps); _fill(c.sigma_w, p.sigma_w)
    c.alpha, c.lam, c.gamma = float(p.alpha), float(p.lam), float(p.gamma)
    c.A, c.B, c.C_u, c.eta = float(p.A), float(p.B), float(p.C_u), float(p.eta)
    _fill(c.nom_p, p.nom_p); _fill(c.risk_p, p.risk_p)
    c.noise_kind = int(getattr(p, "noise_kind", 0))
    _fill(c.noise_p, getattr(p, "noise_p", [0, 0, 0, 0]))
    c.noise_mode = int(getattr(p, "noise_mode", 0))
    c.seed = int(p.seed)
    c.device = int(device)
    c.k_offset = int(getattr(p, "k_offset", 0))
    c.K_total = int(getattr(p, "K_total", 0))
    return c


def make_env(p):
    """Marshal the environment; returns (struct, keepalive arrays)."""
    e = ra_mppi_env()
    keep = []
    if getattr(p, "circles", None) is not None:
        a = np.ascontiguousarray(p.circles, dtype=np.float32)
        keep.append(a)
        e.circles, e.n_circles = a.ctypes.data_as(C.POINTER(C.c_float)), int(a.shape[0])
    if getattr(p, "costmap", None) is not None:
        m = np.ascontiguousarray(p.costmap, dtype=np.float32)
        keep.append(m)
        e.costmap = m.ctypes.data_as(C.POINTER(C.c_float))
        e.map_h, e.map_w = int(m.shape[0]), int(m.shape[1])
        e.map_res, e.map_ox, e.map_oy = float(p.map_res), float(p.map_ox), float(p.map_oy)
    return e, keep


def _check(ctx, st, where):
    if st != RA_OK:
        detail = ""
        if ctx:
            msg = load().ra_mppi_last_error(ctx)
            detail = msg.decode() if msg else ""
        raise RaMppiError(st, where, detail)


# ---- functions with the header's names (pointers are ints: tensor.data_ptr(), stream.cuda_stream)
def ra_mppi_create(cfg: ra_mppi_config, env: ra_mppi_env):
    ctx = C.c_void_p()
    st = load().ra_mppi_create(C.byref(cfg), C.byref(env), C.byref(ctx))
    if st != RA_OK:
        why = load().ra_mppi_create_error()
        raise RaMppiError(st, "ra_mppi_create", why.decode() if why else "")
    return ctx


def ra_mppi_set_env(ctx, env: ra_mppi_env):
    _check(ctx, load().ra_mppi_set_env(ctx, C.byref(env)), "ra_mppi_set_env")


def ra_mppi_step(ctx, d_x0, d_v, iteration, stream=0):
    _check(ctx, load().ra_mppi_step(ctx, d_x0, d_v, int(iteration), stream), "ra_mppi_step")


def ra_mppi_rollout_costs(ctx, d_x0, d_v, iteration, d_S=None, d_cvar=None, d_S_tilde=None, d_L=None,
                          d_xT=None, d_u=None, stream=0):
    _check(ctx, load().ra_mppi_rollout_costs(ctx, d_x0, d_v, int(iteration), d_S, d_cvar, d_S_tilde, d_L,
                                             d_xT, d_u, stream), "ra_mppi_rollout_costs")


def ra_mppi_step_partial(ctx, d_x0, d_v, iteration, d_partial, stream=0):
    _check(ctx, load().ra_mppi_step_partial(ctx, d_x0, d_v, int(iteration), d_partial, stream), "ra_mppi_step_partial")


def ra_mppi_combine_partials(ctx, d_partials, n_parts, d_v_plus, stream=0):
    _check(ctx, load().ra_mppi_combine_partials(ctx, d_partials, int(n_parts), d_v_plus, stream),
           "ra_mppi_combine_partials")


def ra_mppi_weights_update(ctx, d_S_tilde, d_u, d_v_plus, d_w=None, d_stats=None, stream=0):
    _check(ctx, load().ra_mppi_weights_update(ctx, d_S_tilde, d_u, d_v_plus, d_w, d_stats, stream),
           "ra_mppi_weights_update")


RA_STATIC_MAX_K = 131072   # include/ra_mppi.h


def ra_mppi_weights_update_static(K, T, lam, u_min, u_max, d_S_tilde, d_u, d_v_plus, stream=0):
    """Weights (17) and update (4) with no context and no device allocation, for callers that may not call
    cudaMalloc (a loop that gave all its device memory to a fixed pool, a plug-in inside someone else's process,
    a real-time thread): the kernel's scratch is an array compiled into the library.  K <= RA_STATIC_MAX_K,
    T <= 128; the device pointers belong to the CURRENT device.  Calls share that one array, so calls that can
    overlap on the GPU must be ordered by the caller; make the first call on a device outside stream capture."""
    lo, hi = (C.c_float * 2)(*map(float, u_min)), (C.c_float * 2)(*map(float, u_max))
    L = load()
    st = L.ra_mppi_weights_update_static(int(K), int(T), float(lam), lo, hi, d_S_tilde, d_u, d_v_plus, stream)
    if st != RA_OK:
        msg = L.ra_mppi_weights_update_static_error()
        raise RaMppiError(st, "ra_mppi_weights_update_static", msg.decode() if msg else "")


def ra_mppi_step_host(ctx, h_x0, h_v, iteration, stream=0):
    """h_x0, h_v: host addresses (e.g. pinned torch tensor .data_ptr() or numpy .ctypes.data)."""
    _check(ctx, load().ra_mppi_step_host(ctx, h_x0, h_v, int(iteration), stream), "ra_mppi_step_host")


def ra_mppi_enable_kernel_timing(ctx, enable=True):
    _check(ctx, load().ra_mppi_enable_kernel_timing(ctx, 1 if enable else 0), "ra_mppi_enable_kernel_timing")


def ra_mppi_last_rollout_ms(ctx):
    ms = C.c_float()
    _check(ctx, load().ra_mppi_last_rollout_ms(ctx, C.byref(ms)), "ra_mppi_last_rollout_ms")
    return float(ms.value)


def ra_mppi_export_costs_f64(ctx, d_S64=None, d_S_tilde64=None, stream=0):
    _check(ctx, load().ra_mppi_export_costs_f64(ctx, d_S64, d_S_tilde64, stream), "ra_mppi_export_costs_f64")


def ra_mppi_plant_shift(ctx, d_x0, d_v, d_u_applied, iteration, stream=0):
    _check(ctx, load().ra_mppi_plant_shift(ctx, d_x0, d_v, d_u_applied, int(iteration), stream),
           "ra_mppi_plant_shift")


def ra_mppi_closed_loop(ctx, d_x0, d_v, iteration0, n_iter, d_log=None, h_ms=None, stream=0):
    ms_ptr = h_ms.ctypes.data_as(C.POINTER(C.c_float)) if h_ms is not None else None
    _check(ctx, load().ra_mppi_closed_loop(ctx, d_x0, d_v, int(iteration0), int(n_iter), d_log, ms_ptr,
                                           stream), "ra_mppi_closed_loop")


def ra_mppi_philox(ctx, d_ctr, n, d_out, stream=0):
    _check(ctx, load().ra_mppi_philox(ctx, d_ctr, int(n), d_out, stream), "ra_mppi_philox")


def ra_mppi_state_noise(ctx, d_kmt, n, iteration, d_w, stream=0):
    _check(ctx, load().ra_mppi_state_noise(ctx, d_kmt, int(n), int(iteration), d_w, stream),
           "ra_mppi_state_noise")


def ra_mppi_measure_pipe_peaks(device=0):
    """{pipe: 1e12 lane-ops/s} measured by the library's microbenchmark kernels."""
    out = (C.c_float * 4)()
    _check(None, load().ra_mppi_measure_pipe_peaks(int(device), out), "ra_mppi_measure_pipe_peaks")
    return dict(zip(("ffma", "imad_wide", "lop3", "mufu"), (float(x) for x in out)))


def ra_mppi_query_counts(cfg: ra_mppi_config):
    """(k_tail, K0) as ra_mppi_create derives them from the fp32 alpha and eta (host only, no device needed)."""
    k_tail, K0 = C.c_int32(), C.c_int32()
    _check(None, load().ra_mppi_query_counts(C.byref(cfg), C.byref(k_tail), C.byref(K0)), "ra_mppi_query_counts")
    return int(k_tail.value), int(K0.value)


def ra_mppi_rollout_variant(ctx):
    """(dyn, risk, noise variant, slots per lane, half) = the template arguments of the rollout kernel this context launches."""
    out = (C.c_int32 * 5)()
    _check(ctx, load().ra_mppi_rollout_variant(ctx, out), "ra_mppi_rollout_variant")
    return tuple(int(x) for x in out)


def ra_mppi_launches_per_step(ctx):
    return int(load().ra_mppi_launches_per_step(ctx))


def ra_mppi_destroy(ctx):
    if ctx:
        load().ra_mppi_destroy(ctx)
