"""RaMppi: a convenience holder around the C-ABI calls (torch tensors in, torch tensors out).

Allocation and pointer marshalling only -- all arithmetic runs in libra_mppi.so.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B


class RaMppi:
    def __init__(self, problem, device: int = 0):
        if not torch.cuda.is_available():
            raise B.RaMppiError(B.RA_ECUDA, "RaMppi", "no CUDA device: this package has no CPU fallback")
        self.problem = problem
        self.device = torch.device("cuda", device)
        self.cfg = B.make_config(problem, device)
        self.env, self._keep = B.make_env(problem)
        self.ctx = B.ra_mppi_create(self.cfg, self.env)
        self.K, self.M, self.T, self.nx = problem.K, problem.M, problem.T, problem.nx

    def close(self):
        if getattr(self, "ctx", None):
            B.ra_mppi_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_env(self, circles=None, costmap=None, map_res=None, map_ox=None, map_oy=None):
        """ra_mppi_set_env: replace the obstacle set and/or the costmap (same map size) of this controller."""
        kw = {}
        if circles is not None:
            kw["circles"] = np.asarray(circles)
        if costmap is not None:
            kw["costmap"] = np.asarray(costmap)
        for name, val in (("map_res", map_res), ("map_ox", map_ox), ("map_oy", map_oy)):
            if val is not None:
                kw[name] = float(val)
        self.problem = self.problem.replace(**kw)
        self.env, self._keep = B.make_env(self.problem)
        B.ra_mppi_set_env(self.ctx, self.env)

    # ---- helpers
    def tensor(self, a, dtype=torch.float32):
        return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(self.device).contiguous()

    @staticmethod
    def _stream():
        return torch.cuda.current_stream().cuda_stream

    # ---- the C-ABI calls
    def step(self, d_x0: torch.Tensor, d_v: torch.Tensor, iteration: int = 0):
        """In place: d_v [T,2] <- v+ (ra_mppi_step)."""
        assert d_x0.is_cuda and d_v.is_cuda and d_v.dtype == torch.float32 and d_v.is_contiguous()
        B.ra_mppi_step(self.ctx, d_x0.data_ptr(), d_v.data_ptr(), iteration, self._stream())
        return d_v

    def rollout_costs(self, d_x0, d_v, iteration: int = 0, want_L=True, want_xT=True, want_u=True):
        f = dict(device=self.device, dtype=torch.float32)
        out = dict(S=torch.empty(self.K, **f), cvar=torch.empty(self.K, **f), S_tilde=torch.empty(self.K, **f))
        out["L"] = torch.empty(self.K, self.M, **f) if want_L else None
        out["xT"] = torch.empty(self.K, self.M, self.nx, **f) if want_xT else None
        out["u"] = torch.empty(self.K, self.T, 2, **f) if want_u else None
        ptr = lambda t: t.data_ptr() if t is not None else None
        B.ra_mppi_rollout_costs(self.ctx, d_x0.data_ptr(), d_v.data_ptr(), iteration, ptr(out["S"]),
                                ptr(out["cvar"]), ptr(out["S_tilde"]), ptr(out["L"]), ptr(out["xT"]),
                                ptr(out["u"]), self._stream())
        return out

    def step_partial(self, d_x0, d_v, iteration: int = 0, out: torch.Tensor = None):
        """ra_mppi_step_partial: this context's share {beta_g, Z_g, N_g[T,2]} of (17)/(4) as fp64 [2+2T]."""
        if out is None:
            out = torch.empty(2 + 2 * self.T, device=self.device, dtype=torch.float64)
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 2 + 2 * self.T
        B.ra_mppi_step_partial(self.ctx, d_x0.data_ptr(), d_v.data_ptr(), iteration, out.data_ptr(), self._stream())
        return out

    def combine_partials(self, d_partials: torch.Tensor, d_v_out: torch.Tensor = None):
        """ra_mppi_combine_partials: [n, 2+2T] fp64 partials of all shards -> v+ [T,2]."""
        assert d_partials.is_cuda and d_partials.dtype == torch.float64 and d_partials.is_contiguous()
        assert d_partials.dim() == 2 and d_partials.shape[1] == 2 + 2 * self.T
        if d_v_out is None:
            d_v_out = torch.empty(self.T, 2, device=self.device, dtype=torch.float32)
        B.ra_mppi_combine_partials(self.ctx, d_partials.data_ptr(), d_partials.shape[0], d_v_out.data_ptr(),
                                   self._stream())
        return d_v_out

    def step_host(self, h_x0: torch.Tensor, h_v: torch.Tensor, iteration: int = 0):
        """ra_mppi_step_host: h_x0 [nx], h_v [T,2] are HOST tensors (pinned for async copies); h_v <- v+."""
        assert not h_x0.is_cuda and not h_v.is_cuda and h_v.is_contiguous() and h_v.dtype == torch.float32
        B.ra_mppi_step_host(self.ctx, h_x0.data_ptr(), h_v.data_ptr(), iteration, self._stream())
        return h_v

    def enable_kernel_timing(self, enable=True):
        B.ra_mppi_enable_kernel_timing(self.ctx, enable)

    def last_rollout_ms(self):
        return B.ra_mppi_last_rollout_ms(self.ctx)

    def costs_f64(self):
        """fp64 S and S~ of the most recent step / rollout_costs."""
        S = torch.empty(self.K, device=self.device, dtype=torch.float64)
        St = torch.empty(self.K, device=self.device, dtype=torch.float64)
        B.ra_mppi_export_costs_f64(self.ctx, S.data_ptr(), St.data_ptr(), self._stream())
        return S, St

    def weights_update(self, d_S_tilde, d_u):
        f = dict(device=self.device, dtype=torch.float32)
        v_plus, w, stats = torch.empty(self.T, 2, **f), torch.empty(self.K, **f), torch.empty(2, **f)
        B.ra_mppi_weights_update(self.ctx, d_S_tilde.data_ptr(), d_u.data_ptr(), v_plus.data_ptr(),
                                 w.data_ptr(), stats.data_ptr(), self._stream())
        return dict(v_plus=v_plus, w=w, stats=stats)

    def plant_shift(self, d_x0, d_v, iteration: int):
        u = torch.empty(2, device=self.device, dtype=torch.float32)
        B.ra_mppi_plant_shift(self.ctx, d_x0.data_ptr(), d_v.data_ptr(), u.data_ptr(), iteration, self._stream())
        return u

    def closed_loop(self, d_x0, d_v, iteration0: int, n_iter: int, log=True, timing=True):
        d_log = torch.zeros(n_iter, self.nx + 2, device=self.device, dtype=torch.float32) if log else None
        h_ms = np.zeros(n_iter, dtype=np.float32) if timing else None
        B.ra_mppi_closed_loop(self.ctx, d_x0.data_ptr(), d_v.data_ptr(), iteration0, n_iter,
                              d_log.data_ptr() if log else None, h_ms, self._stream())
        return d_log, h_ms

    def philox(self, ctr: torch.Tensor):
        assert ctr.dtype == torch.int64 or ctr.dtype == torch.uint32 or ctr.dtype == torch.int32
        c = ctr.to(torch.int64).to(self.device)
        c32 = (c & 0xFFFFFFFF).to(torch.int64)
        packed = torch.where(c32 >= 2**31, c32 - 2**32, c32).to(torch.int32).contiguous()
        out = torch.empty_like(packed)
        B.ra_mppi_philox(self.ctx, packed.data_ptr(), packed.shape[0], out.data_ptr(), self._stream())
        return out.to(torch.int64) & 0xFFFFFFFF

    def state_noise(self, kmt: torch.Tensor, iteration: int = 0):
        kmt = kmt.to(self.device, torch.int32).contiguous()
        w = torch.empty(kmt.shape[0], self.nx, device=self.device, dtype=torch.float32)
        B.ra_mppi_state_noise(self.ctx, kmt.data_ptr(), kmt.shape[0], iteration, w.data_ptr(), self._stream())
        return w

    @property
    def rollout_variant(self):
        return B.ra_mppi_rollout_variant(self.ctx)

    @property
    def launches_per_step(self):
        return B.ra_mppi_launches_per_step(self.ctx)
