"""Pins P2-P7 of the CPU oracle: closed forms, the exact diagonal case,
brute-force convolution, the dense Lippmann-Schwinger solve and invariants.  CPU only."""
import math

import numpy as np
import pytest
from scipy.special import hankel1

import oracle.tbs_ref as R


def _grid2(N, dx):
    return np.meshgrid(np.arange(N) * dx, np.arange(N) * dx, indexing="ij")  # yy, xx


# ---------------------------------------------------------------- P2: damped closed forms
def _u0_error_2d(ppw):
    """u0 of one point source vs a dx^2 (i/4) H0^(1)(kappa r), kappa = sqrt(k0^2 + i eps)
    (Eq. 16; 2-D form from ref. [32], sign from Alg. 1's G)."""
    lam = 1.5e-3
    dx = lam / ppw
    N = 8 * ppw                      # 8 wavelengths across
    k0, eps = R.wavenumber(1500.0 / lam, 1500.0, 0.8)
    g = R.green_spectrum((2 * N, 2 * N), dx, k0, eps)
    c = N // 2
    S = R.deposit((N, N), dx, [[c * dx, c * dx]], [2.0 - 1.0j])
    u0 = R.apply_G(S, g)
    yy, xx = _grid2(N, dx)
    r = np.hypot(xx - c * dx, yy - c * dx)
    kappa = np.sqrt(k0 ** 2 + 1j * eps)
    assert kappa.imag > 0            # outgoing e^{+i kappa r}, reading A5
    shell = (r > 0.3 * lam) & (r < 2.0 * lam)
    ref = (2.0 - 1.0j) * dx ** 2 * 0.25j * hankel1(0, kappa * r[shell])
    return np.linalg.norm(u0[shell] - ref) / np.linalg.norm(ref)


def test_u0_matches_damped_hankel_2d_and_converges_with_resolution():
    e6, e12, e24 = (_u0_error_2d(p) for p in (6, 12, 24))
    assert e6 < 0.05 and e12 < 0.008 and e24 < 0.0015
    assert e6 / e12 > 3.5 and e12 / e24 > 3.5      # band-limiting error drops ~6x per halving


def test_u0_matches_damped_spherical_wave_3d():
    """3-D: g = exp(i kappa r)/(4 pi r) (ref. [32]); normalisation dx^3."""
    errs = []
    for ppw in (4, 8):
        lam = 1.5e-3
        dx = lam / ppw
        N = 4 * ppw
        k0, eps = R.wavenumber(1500.0 / lam, 1500.0, 0.8)
        g = R.green_spectrum((2 * N,) * 3, dx, k0, eps)
        c = N // 2
        S = R.deposit((N,) * 3, dx, [[c * dx] * 3], [1.0])
        u0 = R.apply_G(S, g)
        ax = np.arange(N) * dx - c * dx
        zz, yy, xx = np.meshgrid(ax, ax, ax, indexing="ij")
        r = np.sqrt(xx ** 2 + yy ** 2 + zz ** 2)
        kappa = np.sqrt(k0 ** 2 + 1j * eps)
        shell = (r > 0.4 * lam) & (r < 1.5 * lam)
        ref = dx ** 3 * np.exp(1j * kappa * r[shell]) / (4 * np.pi * r[shell])
        errs.append(np.linalg.norm(u0[shell] - ref) / np.linalg.norm(ref))
    assert errs[0] < 0.12 and errs[1] < 0.03 and errs[0] / errs[1] > 3.0


# ---------------------------------------------------------------- P3: lossless line source
def test_converged_series_matches_lossless_hankel_sum_with_abl():
    """The converged sum solves the LOSSLESS equation (the -i eps in V undoes the damping,
    PAPER.md:141): p = sum_j a_j dx^2 (i/4) H0^(1)(k0 |r - r_j|) in the interior, provided the
    absorbing layer of Eq. 29 suppresses the crop-edge reflection."""
    N, dx, f, c0 = 128, 0.25e-3, 1.0e6, 1500.0
    k0, eps = R.wavenumber(f, c0, 0.8)
    g = R.green_spectrum((2 * N, 2 * N), dx, k0, eps)
    V = R.potential(np.full((N, N), c0), 0.0, 1.5, f, c0, 0.8)
    cols = np.arange(56, 72)
    pos = np.stack([cols * dx, np.full(16, 40 * dx)], 1)
    amp = np.exp(1j * 0.2 * np.arange(16))
    S = R.deposit((N, N), dx, pos, amp)
    cells = 24
    a = R.abl_window(N, cells)
    res = R.solve(V, S, g, 2000, 1e-9, windows=(a, a))
    assert res.status == R.OK
    yy, xx = _grid2(N, dx)
    ref = np.zeros((N, N), complex)
    for (x, y), aj in zip(pos, amp):
        r = np.hypot(xx - x, yy - y)
        r[r == 0] = 1e-12
        ref += aj * dx ** 2 * 0.25j * hankel1(0, k0 * r)
    m = np.zeros((N, N), bool)
    m[cells + 4:N - cells - 4, cells + 4:N - cells - 4] = True
    m &= np.abs(yy - 40 * dx) > 3 * dx
    err = np.linalg.norm((res.p - ref)[m]) / np.linalg.norm(ref[m])
    assert err < 0.01
    # recorded, not asserted as accuracy: pure crop at damping 0.8 reflects ~18 %
    res0 = R.solve(V, S, g, 2000, 1e-9)
    err0 = np.linalg.norm((res0.p - ref)[m]) / np.linalg.norm(ref[m])
    assert 0.05 < err0 < 0.6


# ---------------------------------------------------------------- P4: exact diagonal case
def test_periodic_homogeneous_series_is_geometric_in_k_space():
    """pad = 1, V == -i eps, A == 1: every operator is diagonal in k-space, so
    p_n^ = S^ g^ (1 - mu^(n+1))/(1 - mu), mu = -i eps g^, and ||u_n||^2 follows by Parseval."""
    N, dx = 32, 0.25e-3
    k0, eps = R.wavenumber(1.0e6, 1500.0, 0.8)
    rng = np.random.default_rng(4)
    S = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    g = R.green_spectrum((N, N), dx, k0, eps)
    V = np.full((N, N), -1j * eps)
    nt = 25
    res = R.solve(V, S, g, nt, 0.0, pad=1)
    assert res.n_terms == nt and res.status == R.NOT_CONVERGED
    # independent evaluation of ghat with numpy's own frequency grid
    kx = 2 * np.pi * np.fft.fftfreq(N, dx)
    gh = 1.0 / (kx[None, :] ** 2 + kx[:, None] ** 2 - k0 ** 2 - 1j * eps)
    assert np.allclose(g, gh, rtol=1e-12)
    Sh = np.fft.fft2(S)
    mu = -1j * eps * gh
    ph = Sh * gh * (1 - mu ** (nt + 1)) / (1 - mu)
    assert np.allclose(res.p, np.fft.ifft2(ph), rtol=1e-10, atol=1e-10 * np.abs(res.p).max())
    for n in (1, 7, nt):
        un2 = np.sum(np.abs(Sh * gh * mu ** n) ** 2) / N ** 2
        pn = np.fft.ifft2(Sh * gh * (1 - mu ** (n + 1)) / (1 - mu))
        assert abs(res.history[n] - math.sqrt(un2) / np.linalg.norm(pn)) < 1e-10
    assert res.history[0] == 1.0


# ---------------------------------------------------------------- P5: brute-force G x
@pytest.mark.parametrize("shape", [(6, 8), (3, 4, 5)])
def test_apply_G_equals_direct_convolution_sum(shape):
    """G x = sum_b g_disc[a - b] x[b] with g_disc = IDFT_M(ghat) by an explicit DFT matrix
    (non-square, non-power-of-two sizes so that a transposed axis or index slip shows)."""
    nd = len(shape)
    dx = 0.3e-3
    k0, eps = R.wavenumber(1.0e6, 1500.0, 0.8)
    M = tuple(2 * s for s in shape)
    g = R.green_spectrum(M, dx, k0, eps)
    gd = g.copy()
    for ax, m in enumerate(M):
        j = np.arange(m)
        Finv = np.exp(2j * np.pi * np.outer(j, j) / m) / m
        gd = np.moveaxis(np.tensordot(Finv, gd, axes=([1], [ax])), 0, ax)
    rng = np.random.default_rng(nd)
    x = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    out = R.apply_G(x, g)
    ref = np.zeros(shape, complex)
    for a in np.ndindex(*shape):
        acc = 0.0
        for b in np.ndindex(*shape):
            idx = tuple((a[i] - b[i]) % M[i] for i in range(nd))
            acc += gd[idx] * x[b]
        ref[a] = acc
    assert np.allclose(out, ref, rtol=1e-11, atol=1e-13 * np.abs(ref).max())
