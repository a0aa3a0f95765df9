"""ctypes binding of the CPU oracle (oracle/tbs_ref.c) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this module.  It never imports the CUDA package and shares no code with it.
All arrays are numpy complex128 / float64, row-major with x fastest (Alg. 1 l.8).
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tbs_ref.c")
_SO = os.path.join(_HERE, "libtbs_ref.so")

OK, NOT_CONVERGED, ERR_INVALID_ARG, ERR_DIVERGED, ERR_ALLOC = 0, 1, -1, -5, -6


def build(force: bool = False) -> str:
    """Compile oracle/tbs_ref.c -> oracle/libtbs_ref.so with gcc (plain C99 + OpenMP)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", _SRC, "-o", _SO, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        L.tbs_ref_num_threads.restype = ctypes.c_int
        L.tbs_ref_fft1d.argtypes = [dp, ctypes.c_int, ctypes.c_int]
        L.tbs_ref_fft1d.restype = None
        L.tbs_ref_green_spectrum.argtypes = [ctypes.c_int, ip, ctypes.c_double, ctypes.c_double,
                                             ctypes.c_double, dp]
        L.tbs_ref_potential.argtypes = [ctypes.c_int64, dp, dp, ctypes.c_double, ctypes.c_double,
                                        ctypes.c_double, ctypes.c_double, ctypes.c_double, dp]
        L.tbs_ref_deposit.argtypes = [ctypes.c_int, ip, ctypes.c_double, ctypes.c_int, dp, dp, dp]
        L.tbs_ref_abl_window.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, dp]
        L.tbs_ref_apply_G.argtypes = [ctypes.c_int, ip, ctypes.c_int, dp, dp, dp]
        L.tbs_ref_solve.argtypes = [ctypes.c_int, ip, ctypes.c_int, dp, dp, dp, dp, dp, dp,
                                    ctypes.c_int, ctypes.c_double, dp, dp, ip, dp]
        L.tbs_ref_second_harmonic_source.argtypes = [ctypes.c_int64, dp, ctypes.c_double,
                                                     ctypes.c_double, ctypes.c_double,
                                                     ctypes.c_double, dp]
        L.tbs_ref_harmonic_source.argtypes = [ctypes.c_int64, ctypes.c_int, ctypes.POINTER(dp), ctypes.c_double,
                                              ctypes.c_double, ctypes.c_double, ctypes.c_double, dp]
        _lib = L
    return _lib


def _dp(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _dims(shape):
    """numpy shape (z, y, x) / (y, x) / (x,) -> ndim and int32 [x, y, z]."""
    nd = len(shape)
    n = np.ones(3, dtype=np.int32)
    for a in range(nd):
        n[a] = shape[nd - 1 - a]
    return nd, n


def num_threads() -> int:
    return int(lib().tbs_ref_num_threads())


def fft1d(x, sign: int):
    """Unnormalised 1-D DFT, X[k] = sum_j x[j] exp(sign 2 pi i jk/n)."""
    a = np.ascontiguousarray(x, dtype=np.complex128).copy()
    lib().tbs_ref_fft1d(_dp(a), a.size, int(sign))
    return a


def wavenumber(f_hz: float, c0: float, damping: float):
    """k0 = 2 pi f/c0 and eps = damping k0^2 (Alg. 1 l.5-6)."""
    k0 = 2.0 * math.pi * f_hz / c0
    return k0, damping * k0 * k0


def green_spectrum(shape_padded, dx: float, k0: float, eps: float):
    nd, m = _dims(shape_padded)
    g = np.empty(shape_padded, dtype=np.complex128)
    rc = lib().tbs_ref_green_spectrum(nd, _ip(m), dx, k0, eps, _dp(g))
    assert rc == OK, rc
    return g


def potential(c, alpha0_db, y: float, f_hz: float, c0: float, damping: float):
    """V = ktilde(r)^2 - k0^2 - i eps; alpha0_db is a scalar or a map shaped like c."""
    c = np.ascontiguousarray(c, dtype=np.float64)
    V = np.empty(c.shape, dtype=np.complex128)
    amap = None
    a0 = 0.0
    if np.ndim(alpha0_db) == 0:
        a0 = float(alpha0_db)
    else:
        amap = np.ascontiguousarray(alpha0_db, dtype=np.float64)
        assert amap.shape == c.shape
    rc = lib().tbs_ref_potential(c.size, _dp(c), _dp(amap), a0, y, f_hz, c0, damping, _dp(V))
    assert rc == OK, rc
    return V


def deposit(shape, dx: float, pos_m, amp):
    nd, n = _dims(shape)
    pos = np.ascontiguousarray(pos_m, dtype=np.float64).reshape(-1, nd)
    a = np.ascontiguousarray(amp, dtype=np.complex128).reshape(-1)
    assert a.size == pos.shape[0]
    S = np.empty(shape, dtype=np.complex128)
    rc = lib().tbs_ref_deposit(nd, _ip(n), dx, pos.shape[0], _dp(pos), _dp(a), _dp(S))
    if rc != OK:
        raise ValueError(f"tbs_ref_deposit failed: {rc}")
    return S


def abl_window(n: int, cells: int, zeta_half_mu: float = 9.666):
    a = np.empty(n, dtype=np.float64)
    rc = lib().tbs_ref_abl_window(n, cells, zeta_half_mu, _dp(a))
    assert rc == OK, rc
    return a


def apply_G(x, ghat, pad: int = 2):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    nd, n = _dims(x.shape)
    ghat = np.ascontiguousarray(ghat, dtype=np.complex128)
    assert ghat.shape == tuple(pad * s for s in x.shape)
    out = np.empty_like(x)
    rc = lib().tbs_ref_apply_G(nd, _ip(n), pad, _dp(ghat), _dp(x), _dp(out))
    assert rc == OK, rc
    return out


@dataclass
class RefResult:
    status: int
    p: np.ndarray
    history: np.ndarray
    n_terms: int
    u_last: np.ndarray


def solve(V, S, ghat, max_terms: int, tol: float, pad: int = 2, windows=None) -> RefResult:
    """Run the term-form Born series.  windows = (ax, ay[, az]) per-axis ABL or None."""
    V = np.ascontiguousarray(V, dtype=np.complex128)
    S = np.ascontiguousarray(S, dtype=np.complex128)
    ghat = np.ascontiguousarray(ghat, dtype=np.complex128)
    assert V.shape == S.shape
    nd, n = _dims(V.shape)
    assert ghat.shape == tuple(pad * s for s in V.shape)
    w = [None, None, None]
    if windows is not None:
        for a in range(nd):
            w[a] = np.ascontiguousarray(windows[a], dtype=np.float64)
            assert w[a].size == n[a]
    p = np.empty_like(V)
    u = np.empty_like(V)
    hist = np.zeros(max_terms + 1, dtype=np.float64)
    nt = np.zeros(1, dtype=np.int32)
    rc = lib().tbs_ref_solve(nd, _ip(n), pad, _dp(ghat), _dp(V), _dp(S), _dp(w[0]), _dp(w[1]),
                             _dp(w[2]), int(max_terms), float(tol), _dp(p), _dp(hist), _ip(nt),
                             _dp(u))
    if rc < 0 and rc != ERR_DIVERGED:
        raise RuntimeError(f"tbs_ref_solve failed: {rc}")
    k = int(nt[0])
    return RefResult(int(rc), p, hist[: k + 1].copy(), k, u)


def second_harmonic_source(p1, beta: float, rho0: float, c0: float, f1_hz: float):
    p1 = np.ascontiguousarray(p1, dtype=np.complex128)
    S2 = np.empty_like(p1)
    rc = lib().tbs_ref_second_harmonic_source(p1.size, _dp(p1), beta, rho0, c0, f1_hz, _dp(S2))
    assert rc == OK, rc
    return S2


def harmonic_source(h: int, fields, beta: float, rho0: float, c0: float, f1_hz: float):
    """S_h of Eqs. 28b-28e from the fields of harmonics 1..h-1 (`fields[m]` = psi_{m+1})."""
    fs = [np.ascontiguousarray(f, dtype=np.complex128) for f in fields[:h - 1]]
    assert len(fs) == h - 1
    S = np.empty_like(fs[0])
    dp = ctypes.POINTER(ctypes.c_double)
    ptrs = (dp * 4)(*([_dp(f) for f in fs] + [None] * (4 - len(fs))))
    rc = lib().tbs_ref_harmonic_source(fs[0].size, int(h), ptrs, beta, rho0, c0, f1_hz, _dp(S))
    assert rc == OK, rc
    return S


def solve_cbs(V, S, ghat, eps_nd: float, max_terms: int, tol: float, pad: int = 2, windows=None) -> RefResult:
    """Convergent Born series (PAPER.md:25, 445, 475 name it, its ref. [16] defines it):
    preconditioner gamma = i V / eps, psi <- psi + gamma (G(V psi + S) - psi).  In term form, with
    M = gamma G V + 1 - gamma:   u_0 = gamma A G S,   u_{n+1} = (1 - gamma) u_n + gamma A G(V u_n),   p = sum u_n.
    V and eps_nd in the same units (both divided by k0^2, or both not).  Plain numpy on top of apply_G;
    stopping rule and history as in solve().  For V = -i eps (homogeneous, lossless) gamma = 1 and the
    iterates are those of the traditional series."""
    V = np.ascontiguousarray(V, dtype=np.complex128)
    S = np.ascontiguousarray(S, dtype=np.complex128)
    A = np.ones(V.shape)
    if windows is not None:
        nd = V.ndim
        for a in range(nd):
            shp = [1] * nd
            shp[nd - 1 - a] = -1
            A = A * np.asarray(windows[a], dtype=np.float64).reshape(shp)
    gamma = 1j * V / eps_nd
    u = gamma * (A * apply_G(S, ghat, pad))
    p = u.copy()
    hist = [1.0]
    status, k = NOT_CONVERGED, 0
    if max_terms == 0:
        return RefResult(status, p, np.array(hist), 0, u)
    for k in range(1, max_terms + 1):
        u = (1.0 - gamma) * u + gamma * (A * apply_G(V * u, ghat, pad))
        p += u
        r = math.sqrt(float(np.vdot(u, u).real)) / math.sqrt(float(np.vdot(p, p).real))
        hist.append(r)
        if not math.isfinite(r):
            status = ERR_DIVERGED
            break
        if r < tol:
            status = OK
            break
    return RefResult(status, p, np.array(hist), k, u)


def solve_paper_mode(V, S, ghat_periodic, max_iter: int, tol: float, row: int, windows=None) -> RefResult:
    """Algorithm 1 l.36-47 as printed, in the paper's own Picard form on the periodic
    N-grid (pad factor 1):  psi_in = A G S;  psi_fn = A G(V psi_in + S);  error = sum_m |psi_fn(row, m) -
    psi_in(row, m)| / sum_m |psi_in(row, m)| (Eq. 30);  stop at the first error < tol.
    Reading A4: the window multiplies the initial field too.  history[l] = error of iteration l, n_terms =
    iterations done.  Rows are indexed as the flattened slow axes (y in 2-D, z*ny + y in 3-D)."""
    V = np.ascontiguousarray(V, dtype=np.complex128)
    S = np.ascontiguousarray(S, dtype=np.complex128)
    A = np.ones(V.shape)
    if windows is not None:
        nd = V.ndim
        for a in range(nd):
            shp = [1] * nd
            shp[nd - 1 - a] = -1
            A = A * np.asarray(windows[a], dtype=np.float64).reshape(shp)
    nx = V.shape[-1]
    psi = A * apply_G(S, ghat_periodic, 1)
    hist = [1.0]
    status, l = NOT_CONVERGED, 0
    for l in range(1, max_iter + 1):
        new = A * apply_G(V * psi + S, ghat_periodic, 1)
        err = float(np.abs(new.reshape(-1, nx)[row] - psi.reshape(-1, nx)[row]).sum()
                    / np.abs(psi.reshape(-1, nx)[row]).sum())
        u = new - psi
        psi = new
        hist.append(err)
        if not math.isfinite(err):
            status = ERR_DIVERGED
            break
        if err < tol:
            status = OK
            break
    return RefResult(status, psi, np.array(hist), l, u if max_iter > 0 else psi)


def kspace_potential(shape_padded, dx: float, alpha0_si: float, nu: float, f_hz: float, c0: float, damping: float,
                     dispersive: bool = True):
    """VV(k) = -i tau w k^nu + eta k^(nu+1) - i eps on the FFT grid (Eq. 24; Alg. 1 l.23,
    PAPER.md:323), tau = -2 alpha0 v_f^(nu-1), eta = 2 alpha0 v_f^nu tan(pi nu/2), k = |p|."""
    w = 2.0 * math.pi * f_hz
    k0, eps = wavenumber(f_hz, c0, damping)
    tau = -2.0 * alpha0_si * c0 ** (nu - 1.0)
    eta = 2.0 * alpha0_si * c0 ** nu * math.tan(math.pi * nu / 2.0) if dispersive else 0.0
    k2 = np.zeros(shape_padded)
    nd = len(shape_padded)
    for ax, m in enumerate(shape_padded):
        p = 2.0 * math.pi * np.fft.fftfreq(m, d=dx)
        shp = [1] * nd
        shp[ax] = m
        k2 = k2 + (p ** 2).reshape(shp)
    k = np.sqrt(k2)
    return -1j * tau * w * k ** nu + eta * k ** (nu + 1.0) - 1j * eps


def solve_kspace(S, ghat, VV, max_terms: int, tol: float, pad: int = 2, windows=None, row=None, Us=None) -> RefResult:
    """Eq. 24 in term form: u_0 = A G S, u_{n+1} = A F^-1[ghat VV F[u_n]], p = sum u_n (the Picard iterates of
    Eq. 24 are these partial sums).  row = None: r_n = ||u_n||_2/||p_n||_2; row = r: Eq. 30 on that row.
    Us (optional, same shape as S): a scatterer in the absorbing medium -- the potential of Eq. 23
    plus the spatial term U_s(r) = k_s(r)^2 - k_f^2 of Eq. 25 (the -i eps is already in VV):
    u_{n+1} = A F^-1[ghat (VV F[u_n] + F[U_s u_n])].  The paper runs the two potentials separately (Eq. 24, Eq. 26);
    this is their sum, both being terms of the same operator V in psi = G V psi + G S (Eq. 17)."""
    S = np.ascontiguousarray(S, dtype=np.complex128)
    A = np.ones(S.shape)
    if windows is not None:
        nd = S.ndim
        for a in range(nd):
            shp = [1] * nd
            shp[nd - 1 - a] = -1
            A = A * np.asarray(windows[a], dtype=np.float64).reshape(shp)
    nx = S.shape[-1]
    gv = np.ascontiguousarray(ghat * VV)
    u = A * apply_G(S, ghat, pad)
    p = u.copy()
    hist = [1.0]
    status, k = NOT_CONVERGED, 0
    for k in range(1, max_terms + 1):
        if Us is None:
            u = A * apply_G(u, gv, pad)
        else:
            u = A * (apply_G(u, gv, pad) + apply_G(Us * u, ghat, pad))
        if row is None:
            p += u
            r = math.sqrt(float(np.vdot(u, u).real)) / math.sqrt(float(np.vdot(p, p).real))
        else:
            r = float(np.abs(u.reshape(-1, nx)[row]).sum() / np.abs(p.reshape(-1, nx)[row]).sum())
            p += u
        hist.append(r)
        if not math.isfinite(r):
            status = ERR_DIVERGED
            break
        if r < tol:
            status = OK
            break
    return RefResult(status, p, np.array(hist), k, u)
