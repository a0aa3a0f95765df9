"""Thin Python binding of the C ABI in include/tbs.h -- argument marshalling only.

Every step of the Born-series path runs in the CUDA kernels of libtbs.so; torch is used here for
device memory and streams, nothing else.  Names follow the C entry points (``tbs_*``).
Arrays are (y, x) / (z, y, x) with x fastest; complex fields are torch.complex64 on the device.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass

import numpy as np
import torch

from . import _lib

OK, NOT_CONVERGED = 0, 1
ERR_INVALID_ARG, ERR_UNSUPPORTED_SIZE, ERR_NOT_READY, ERR_CUDA, ERR_DIVERGED, ERR_ALLOC = -1, -2, -3, -4, -5, -6


class TbsError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"tbs status {status}: {msg}")
        self.status = status


@dataclass
class SolveResult:
    status: int            # OK, NOT_CONVERGED or ERR_DIVERGED
    p: "torch.Tensor | np.ndarray"   # [nfreq, *shape] complex64 (device tensor, or host array for solve_host)
    history: np.ndarray    # [nfreq, max_terms+1] float64, history[k] = ||u_k||/||p_k||
    n_terms: np.ndarray    # [nfreq] int32
    loop_ms: float         # device time of the term loops (CUDA events)
    launches: int          # kernels launched by the solve


def _stream_ptr():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev_ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else None


class Plan:
    """tbs_plan: one grid x nfreq frequencies."""

    def __init__(self, shape, dx, freqs, c0, damping=0.8):
        self._L = _lib.load()
        self._h = ctypes.c_void_p()
        self.shape = tuple(int(s) for s in shape)
        self.ndim = len(self.shape)
        self.freqs = [float(f) for f in np.atleast_1d(freqs)]
        self.nfreq = len(self.freqs)
        self.dx, self.c0, self.damping = float(dx), float(c0), float(damping)
        n = np.ones(3, dtype=np.int32)
        for a in range(self.ndim):
            n[a] = self.shape[self.ndim - 1 - a]
        f = np.asarray(self.freqs, dtype=np.float64)
        st = self._L.tbs_plan_create(ctypes.byref(self._h), self.ndim,
                                     n.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), self.dx, self.nfreq,
                                     f.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), self.c0, self.damping)
        if st != OK:
            self._h = ctypes.c_void_p()
            raise TbsError(st, "tbs_plan_create failed")
        self.npts = int(np.prod(self.shape))

    # ------------------------------------------------------------------ helpers
    def _check(self, st, allow=(OK,)):
        if st not in allow:
            raise TbsError(st, self._L.tbs_last_error(self._h).decode())
        return st

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._L.tbs_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _field(self, t, name):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex64 and t.is_contiguous()
                and tuple(t.shape) == self.shape):
            raise ValueError(f"{name}: expected a contiguous CUDA complex64 tensor of shape {self.shape}")
        return t

    def _map(self, t, name):
        if t is None:
            return None
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                and tuple(t.shape) == self.shape):
            raise ValueError(f"{name}: expected a contiguous CUDA float32 tensor of shape {self.shape}")
        return t

    # ------------------------------------------------------------------ C ABI, one method per call
    def workspace_bytes(self):
        """tbs_plan_workspace_bytes: size of the workspace the plan needs (known before anything is allocated)."""
        return int(self._L.tbs_plan_workspace_bytes(self._h))

    def set_workspace(self, buf):
        """tbs_plan_set_workspace: run in a caller-owned CUDA tensor (any dtype, contiguous, >= workspace_bytes()).
        The plan keeps a reference so the memory outlives it."""
        if not (isinstance(buf, torch.Tensor) and buf.is_cuda and buf.is_contiguous()):
            raise ValueError("workspace: expected a contiguous CUDA tensor")
        self._check(self._L.tbs_plan_set_workspace(self._h, ctypes.c_void_p(buf.data_ptr()),
                                                   buf.numel() * buf.element_size()))
        self._ws = buf

    def device_bytes(self):
        return int(self._L.tbs_plan_device_bytes(self._h))

    def set_launch_overlap(self, on):
        """tbs_set_launch_overlap: programmatic dependent launch of the term kernels (default on)."""
        self._check(self._L.tbs_set_launch_overlap(self._h, int(bool(on))))

    def set_concurrency(self, members):
        """tbs_set_concurrency: members of a frequency batch solved at once (1 or 2)."""
        self._check(self._L.tbs_set_concurrency(self._h, int(members)))

    def set_scheme(self, scheme):
        """tbs_set_scheme: "born" (traditional series, default) or "cbs" (convergent Born series)."""
        code = {"born": 0, "tbs": 0, "cbs": 1}[scheme] if isinstance(scheme, str) else int(scheme)
        self._check(self._L.tbs_set_scheme(self._h, code))

    def set_kspace_absorption(self, alpha0_si, nu, dispersive=True):
        """tbs_set_kspace_absorption: homogeneous power-law medium as the k-space multiplier of Eq. 24."""
        self._check(self._L.tbs_set_kspace_absorption(self._h, float(alpha0_si), float(nu), int(bool(dispersive))))

    def set_kspace_scatterer(self, c):
        """tbs_set_kspace_scatterer: a sound-speed map next to the k-space multiplier (periodic boundary, 2-D)."""
        self._check(self._L.tbs_set_kspace_scatterer(self._h, _dev_ptr(self._map(c, "c")), _stream_ptr()))

    def set_boundary(self, boundary):
        """tbs_set_boundary: "pad" (zero-pad/crop, default) or "periodic" (the paper's N-grid FFTs)."""
        code = {"pad": 0, "periodic": 1}[boundary] if isinstance(boundary, str) else int(boundary)
        self._check(self._L.tbs_set_boundary(self._h, code))

    def set_criterion(self, criterion, row=0):
        """tbs_set_criterion: "l2_grid" (default) or "l1_row" (Eq. 30 of the paper on grid row `row`)."""
        code = {"l2_grid": 0, "l1_row": 1}[criterion] if isinstance(criterion, str) else int(criterion)
        self._check(self._L.tbs_set_criterion(self._h, code, int(row)))

    def set_abl(self, cells, zeta_half_mu=9.666):
        self._check(self._L.tbs_set_abl(self._h, int(cells), float(zeta_half_mu)))

    def set_graph_batch(self, terms_per_graph):
        self._check(self._L.tbs_set_graph_batch(self._h, int(terms_per_graph)))

    def set_medium(self, c, rho=None, alpha0_map=None, alpha0_db=0.0, y=1.5, beta=1.0, rho0=1000.0):
        c, rho, alpha0_map = self._map(c, "c"), self._map(rho, "rho"), self._map(alpha0_map, "alpha0_map")
        self._check(self._L.tbs_set_medium(self._h, _dev_ptr(c), _dev_ptr(rho), _dev_ptr(alpha0_map),
                                           float(alpha0_db), float(y), float(beta), float(rho0), _stream_ptr()))

    def set_medium_host(self, c, rho=None, alpha0_map=None, alpha0_db=0.0, y=1.5, beta=1.0, rho0=1000.0):
        def hp(a, name):
            if a is None:
                return None
            if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous
                    and a.shape == self.shape):
                raise ValueError(f"{name}: expected a C-contiguous float32 numpy array of shape {self.shape}")
            return ctypes.c_void_p(a.ctypes.data)
        self._check(self._L.tbs_set_medium_host(self._h, hp(c, "c"), hp(rho, "rho"), hp(alpha0_map, "alpha0_map"),
                                                float(alpha0_db), float(y), float(beta), float(rho0),
                                                _stream_ptr()))

    def set_potential(self, ifreq, V):
        self._check(self._L.tbs_set_potential(self._h, int(ifreq), _dev_ptr(self._field(V, "V")), _stream_ptr()))

    def set_source(self, pos_m, amp):
        pos = np.ascontiguousarray(pos_m, dtype=np.float64).reshape(-1, self.ndim)
        a = np.ascontiguousarray(amp, dtype=np.complex64).reshape(self.nfreq, -1)
        if a.shape[1] != pos.shape[0]:
            raise ValueError("amp must be [nfreq][n_src]")
        self._check(self._L.tbs_set_source(self._h, pos.shape[0],
                                           pos.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                           a.view(np.float32).ctypes.data_as(ctypes.POINTER(ctypes.c_float)),
                                           _stream_ptr()))

    def set_source_field(self, ifreq, S):
        self._check(self._L.tbs_set_source_field(self._h, int(ifreq), _dev_ptr(self._field(S, "S")), _stream_ptr()))

    def _outs(self, max_terms):
        hist = np.zeros((self.nfreq, max_terms + 1), dtype=np.float64)
        nt = np.zeros(self.nfreq, dtype=np.int32)
        return hist, nt

    def solve(self, max_terms, tol, out=None) -> SolveResult:
        p = out if out is not None else torch.empty((self.nfreq,) + self.shape, dtype=torch.complex64, device="cuda")
        hist, nt = self._outs(max_terms)
        st = self._L.tbs_solve(self._h, int(max_terms), float(tol), _dev_ptr(p),
                               hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                               nt.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _stream_ptr())
        self._check(st, allow=(OK, NOT_CONVERGED, ERR_DIVERGED))
        return SolveResult(st, p, hist, nt, self.last_loop_ms(), self.last_launch_count())

    def solve_resume(self, max_terms, tol, out=None) -> SolveResult:
        """tbs_solve_resume: continue the series the last solve() left at its cap, up to max_terms terms in all."""
        p = out if out is not None else torch.empty((self.nfreq,) + self.shape, dtype=torch.complex64, device="cuda")
        hist, nt = self._outs(max_terms)
        st = self._L.tbs_solve_resume(self._h, int(max_terms), float(tol), _dev_ptr(p),
                                      hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                      nt.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _stream_ptr())
        self._check(st, allow=(OK, NOT_CONVERGED, ERR_DIVERGED))
        return SolveResult(st, p, hist, nt, self.last_loop_ms(), self.last_launch_count())

    def solve_host(self, max_terms, tol, out=None) -> SolveResult:
        p = out if out is not None else np.empty((self.nfreq,) + self.shape, dtype=np.complex64)
        hist, nt = self._outs(max_terms)
        st = self._L.tbs_solve_host(self._h, int(max_terms), float(tol), ctypes.c_void_p(p.ctypes.data),
                                    hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                    nt.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _stream_ptr())
        self._check(st, allow=(OK, NOT_CONVERGED, ERR_DIVERGED))
        return SolveResult(st, p, hist, nt, self.last_loop_ms(), self.last_launch_count())

    def apply_green(self, ifreq, x):
        out = torch.empty_like(self._field(x, "x"))
        self._check(self._L.tbs_apply_green(self._h, int(ifreq), _dev_ptr(x), _dev_ptr(out), _stream_ptr()))
        return out

    def get_potential(self, ifreq):
        out = torch.empty(self.shape, dtype=torch.complex64, device="cuda")
        self._check(self._L.tbs_get_potential(self._h, int(ifreq), _dev_ptr(out), _stream_ptr()))
        return out

    def get_source(self, ifreq):
        out = torch.empty(self.shape, dtype=torch.complex64, device="cuda")
        self._check(self._L.tbs_get_source(self._h, int(ifreq), _dev_ptr(out), _stream_ptr()))
        return out

    def green_spectrum(self, ifreq):
        out = torch.empty(tuple(2 * s for s in self.shape), dtype=torch.complex64, device="cuda")
        self._check(self._L.tbs_green_spectrum(self._h, int(ifreq), _dev_ptr(out), _stream_ptr()))
        return out

    def last_launch_count(self):
        return int(self._L.tbs_last_launch_count(self._h))

    def last_loop_ms(self):
        return float(self._L.tbs_last_loop_ms(self._h))

    def profile_term(self, ifreq=0, reps=20):
        ms = np.zeros(4, dtype=np.float64)
        self._check(self._L.tbs_profile_term(self._h, int(ifreq), int(reps),
                                             ms.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), _stream_ptr()))
        return ms


def solve_second_harmonic(plan1: Plan, plan2: Plan, max_terms, tol, ref_row, surface_pressure_pa):
    """tbs_solve_second_harmonic: returns (status, (SolveResult for f1, SolveResult for 2 f1))."""
    L = plan1._L
    p1 = torch.empty((1,) + plan1.shape, dtype=torch.complex64, device="cuda")
    p2 = torch.empty((1,) + plan2.shape, dtype=torch.complex64, device="cuda")
    h1, n1 = plan1._outs(max_terms)
    h2, n2 = plan2._outs(max_terms)
    dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
    st = L.tbs_solve_second_harmonic(plan1._h, plan2._h, int(max_terms), float(tol), int(ref_row),
                                     float(surface_pressure_pa), _dev_ptr(p1), _dev_ptr(p2),
                                     h1.ctypes.data_as(dp), h2.ctypes.data_as(dp), n1.ctypes.data_as(ip),
                                     n2.ctypes.data_as(ip), _stream_ptr())
    if st not in (OK, NOT_CONVERGED, ERR_DIVERGED):
        raise TbsError(st, L.tbs_last_error(plan2._h).decode() or L.tbs_last_error(plan1._h).decode())
    r1 = SolveResult(st, p1, h1, n1, plan1.last_loop_ms(), plan1.last_launch_count())
    r2 = SolveResult(st, p2, h2, n2, plan2.last_loop_ms(), plan2.last_launch_count())
    return st, (r1, r2)


def solve_harmonics(plans, max_terms, tol, ref_row, surface_pressure_pa):
    """tbs_solve_harmonics: plans[h-1] created at h*f1; returns (status, [SolveResult per harmonic])."""
    L = plans[0]._L
    nh = len(plans)
    vp, dp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
    outs = [torch.empty((1,) + pl.shape, dtype=torch.complex64, device="cuda") for pl in plans]
    hists = [np.zeros((1, max_terms + 1), dtype=np.float64) for _ in plans]
    nt = np.zeros(nh, dtype=np.int32)
    h_arr = (vp * nh)(*[pl._h for pl in plans])
    o_arr = (vp * nh)(*[vp(o.data_ptr()) for o in outs])
    hi_arr = (dp * nh)(*[h.ctypes.data_as(dp) for h in hists])
    st = L.tbs_solve_harmonics(h_arr, nh, int(max_terms), float(tol), int(ref_row), float(surface_pressure_pa),
                               o_arr, hi_arr, nt.ctypes.data_as(ip), _stream_ptr())
    if st not in (OK, NOT_CONVERGED, ERR_DIVERGED):
        msgs = [L.tbs_last_error(pl._h).decode() for pl in plans]
        raise TbsError(st, next((m for m in msgs if m), ""))
    res = [SolveResult(st, outs[i], hists[i], nt[i:i + 1].copy(), plans[i].last_loop_ms(), plans[i].last_launch_count())
           for i in range(nh)]
    return st, res


def grid_harmonic_frequency(m, c0, n, dx):
    """tbs_grid_harmonic_frequency: the m-th frequency a periodic n-point grid carries exactly."""
    return float(_lib.load().tbs_grid_harmonic_frequency(int(m), float(c0), int(n), float(dx)))
