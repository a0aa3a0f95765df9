"""Pins of the oracle's convergent Born series.  The paper names the scheme and its
convergence condition and leaves the formula to its ref. [16]; what pins the oracle
here is mathematics, not that reference: the fixed point is the solution of the same linear system as the
traditional series (dense direct solve), the iteration matrix is M = gamma G V + 1 - gamma, and for a
homogeneous lossless medium gamma = 1 makes the two schemes identical.  CPU only."""
import numpy as np

import oracle.tbs_ref as R
from test_oracle_pins_c import _dense_G


def _strong_problem(N, ratio):
    """Large slow disc: k^2/k0^2 - 1 = ratio^2 - 1 inside (below the damping 0.8 for ratio < 1.34)."""
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / 6.0
    ax = np.arange(N) - (N - 1) / 2
    yy, xx = np.meshgrid(ax, ax, indexing="ij")
    c = np.full((N, N), c0)
    c[np.hypot(xx, yy) < N / 3] = c0 / ratio
    V = R.potential(c, 0.0, 1.5, f, c0, 0.8)
    k0, eps = R.wavenumber(f, c0, 0.8)
    g = R.green_spectrum((2 * N, 2 * N), dx, k0, eps)
    S = np.zeros((N, N), complex)
    S[1, 1] = 1.0
    S[2, N // 2] = 0.5j
    return V, S, g, eps


def test_cbs_equals_tbs_for_homogeneous_lossless_medium():
    """V = -i eps  =>  gamma = i V / eps = 1  =>  M = G V: same terms, same history."""
    N = 24
    V, S, g, eps = _strong_problem(N, 1.0)
    assert np.allclose(V, -1j * eps)
    a = R.solve(V, S, g, 60, 0.0)
    b = R.solve_cbs(V, S, g, eps, 60, 0.0)
    assert np.abs(a.p - b.p).max() < 1e-12 * np.abs(a.p).max()
    assert np.allclose(a.history, b.history, rtol=1e-10)


def test_cbs_converges_to_the_dense_solution_where_the_traditional_series_diverges():
    """eps >= max |k^2 - k0^2| is enough for CBS; the same medium has rho(G V) > 1."""
    N = 16
    V, S, g, eps = _strong_problem(N, 1.3)
    assert np.abs(V + 1j * eps).max() <= eps          # |k^2 - k0^2| <= eps
    n = N * N
    G = _dense_G(g, (N, N))
    GV = G * V.reshape(1, n)
    assert np.abs(np.linalg.eigvals(GV)).max() > 1.0  # the traditional series diverges
    tbs = R.solve(V, S, g, 400, 1e-12)
    assert tbs.status != R.OK
    p_dense = np.linalg.solve(np.eye(n) - GV, G @ S.reshape(n)).reshape(N, N)
    res = R.solve_cbs(V, S, g, eps, 20000, 1e-13)
    assert res.status == R.OK
    assert np.linalg.norm(res.p - p_dense) < 1e-9 * np.linalg.norm(p_dense)
    # iteration matrix M = gamma G V + 1 - gamma: contraction, and its spectral radius is the tail ratio
    gam = (1j * V / eps).reshape(n)
    M = gam[:, None] * GV + np.diag(1.0 - gam)
    rho = np.abs(np.linalg.eigvals(M)).max()
    assert rho < 1.0
    h, k = res.history, res.n_terms
    assert abs(h[k] / h[k - 1] - rho) < 2e-2


def test_cbs_first_terms_follow_the_definition():
    """u_0 = gamma G S, u_1 = (1 - gamma) u_0 + gamma G(V u_0), written out with the dense matrix."""
    N = 12
    V, S, g, eps = _strong_problem(N, 1.2)
    n = N * N
    G = _dense_G(g, (N, N))
    gam = (1j * V / eps).reshape(n)
    u0 = gam * (G @ S.reshape(n))
    u1 = (1 - gam) * u0 + gam * (G @ (V.reshape(n) * u0))
    res = R.solve_cbs(V, S, g, eps, 1, 0.0)
    assert np.abs(res.p.reshape(n) - (u0 + u1)).max() < 1e-12 * np.abs(u0).max()
    assert abs(res.history[1] - np.linalg.norm(u1) / np.linalg.norm(u0 + u1)) < 1e-12


# ---------------------------------------------------------------- paper mode
def test_paper_mode_equals_algorithm_1_written_with_numpy_fft():
    """Alg. 1 l.36-44 typed with numpy's FFT (a library routine, not the oracle's own):
    periodic N-grid, window after every iteration, error of Eq. 30 on one row."""
    N, f, c0 = 48, 1.0e6, 1500.0
    dx = c0 / f / 6.0
    k0, eps = R.wavenumber(f, c0, 0.8)
    rng = np.random.default_rng(3)
    c = c0 * (1 + 0.02 * rng.standard_normal((N, N)))
    V = R.potential(c, 0.0, 1.5, f, c0, 0.8)
    S = np.zeros((N, N), complex)
    S[20:28, 10] = -1.0e6j                       # Alg. 1 l.15: S = (0, -10^6) on the source pixels
    g = R.green_spectrum((N, N), dx, k0, eps)
    win = tuple(R.abl_window(N, 10) for _ in range(2))
    A = win[1][:, None] * win[0][None, :]
    res = R.solve_paper_mode(V, S, g, 25, 0.0, N // 2, windows=win)
    psi = A * np.fft.ifft2(g * np.fft.fft2(S))
    errs = []
    for _ in range(25):
        new = A * np.fft.ifft2(g * np.fft.fft2(V * psi + S))
        errs.append(np.abs(new[N // 2] - psi[N // 2]).sum() / np.abs(psi[N // 2]).sum())
        psi = new
    assert np.abs(res.p - psi).max() < 1e-10 * np.abs(psi).max()
    assert np.allclose(res.history[1:], errs, rtol=1e-9)


def test_paper_mode_partial_sums_are_the_term_form_with_pad_factor_one():
    """The Picard iterates on the periodic grid are the partial sums of the term form (Eq. 18 vs Eq. 19)."""
    N, f, c0 = 32, 1.0e6, 1500.0
    dx = c0 / f / 6.0
    k0, eps = R.wavenumber(f, c0, 0.8)
    c = np.full((N, N), c0)
    c[10:20, 12:22] = 1560.0
    V = R.potential(c, 0.5, 1.1, f, c0, 0.8)
    S = np.zeros((N, N), complex)
    S[5, 8:24] = 1.0
    g = R.green_spectrum((N, N), dx, k0, eps)
    win = tuple(R.abl_window(N, 6) for _ in range(2))
    a = R.solve_paper_mode(V, S, g, 12, 0.0, N // 2, windows=win)
    b = R.solve(V, S, g, 12, 0.0, pad=1, windows=win)
    assert np.abs(a.p - b.p).max() < 1e-12 * np.abs(b.p).max()


# ---------------------------------------------------------------- k-space multiplier potential (Eq. 24)
def _kspace_case(ny, nx, ppw=8.0):
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / ppw
    return f, c0, dx


def test_kspace_potential_on_shell_value_and_printed_constants(golden):
    """VV(k_f) + i eps = k_f^nu (eta k_f - i tau w) = 2 k_f alpha (tan(pi nu/2) + i), alpha = alpha0 w^nu (Eq. 3,
    PAPER.md:51): the multiplier reproduces the power law on shell; tau, eta as printed in Table 4."""
    f, c0 = golden["f_hz"], golden["v_f"]
    a0, nu = golden["alpha0_si"], golden["nu"]
    w = 2 * np.pi * f
    k0, eps = R.wavenumber(f, c0, 0.8)
    M = 64
    dx = 2 * np.pi / (M * k0) * 8          # so that bin 8 of the FFT grid sits exactly on |p| = k0
    VV = R.kspace_potential((M,), dx, a0, nu, f, c0, 0.8)
    on_shell = VV[8] + 1j * eps
    alpha = a0 * w ** nu
    expect = 2 * k0 * alpha * (np.tan(np.pi * nu / 2) + 1j)
    assert abs(on_shell - expect) < 1e-9 * abs(expect)
    tau = -2 * a0 * c0 ** (nu - 1)
    eta = 2 * a0 * c0 ** nu * np.tan(np.pi * nu / 2)
    assert abs(tau / golden["tau"] - 1) < 0.02 and abs(eta / golden["eta"] - 1) < 0.02


def test_kspace_series_equals_equation_24_typed_with_numpy_fft():
    f, c0, dx = _kspace_case(32, 32)
    N = 40
    k0, eps = R.wavenumber(f, c0, 0.8)
    a0, nu = 8.0e-9, 1.5
    g = R.green_spectrum((N, N), dx, k0, eps)
    VV = R.kspace_potential((N, N), dx, a0, nu, f, c0, 0.8)
    S = np.zeros((N, N), complex)
    S[14:26, 8] = -1.0e6j
    win = tuple(R.abl_window(N, 8) for _ in range(2))
    A = win[1][:, None] * win[0][None, :]
    res = R.solve_kspace(S, g, VV, 20, 0.0, pad=1, windows=win, row=N // 2)
    psi = A * np.fft.ifft2(g * np.fft.fft2(S))
    errs = []
    for _ in range(20):                     # Eq. 24 as printed, Picard form, window after every iteration
        new = A * np.fft.ifft2(g * (VV * np.fft.fft2(psi) + np.fft.fft2(S)))
        errs.append(np.abs(new[N // 2] - psi[N // 2]).sum() / np.abs(psi[N // 2]).sum())
        psi = new
    assert np.abs(res.p - psi).max() < 1e-10 * np.abs(psi).max()
    assert np.allclose(res.history[1:], errs, rtol=1e-8)


def test_kspace_series_plane_wave_decays_with_the_power_law():
    """A source uniform in y on a grid periodic in y radiates plane waves along x; between two planes their
    amplitude and phase must follow the complex wavenumber of the absorbing-dispersive wave equation (Eq. 7)."""
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / 8.0
    ny, nx = 4, 1024
    k0, eps = R.wavenumber(f, c0, 0.8)
    a0, nu = 6.0e-9, 1.5                      # alpha = a0 w^nu ~ 94 Np/m: e^-1 over ~57 cells
    g = R.green_spectrum((ny, nx), dx, k0, eps)
    VV = R.kspace_potential((ny, nx), dx, a0, nu, f, c0, 0.8)
    S = np.zeros((ny, nx), complex)
    S[:, 200] = 1.0
    win = (R.abl_window(nx, 150), np.ones(ny))
    res = R.solve_kspace(S, g, VV, 3000, 1e-10, pad=1, windows=win)
    assert res.status == R.OK
    a, b = 300, 700
    # plane wave e^{iKx} in Eq. 7: K^2 = k_f^2 - i tau w K^nu + eta K^(nu+1); to first order in
    # alpha/k this is K = k_f + alpha (tan(pi nu/2) + i) with alpha = alpha0 w^nu (Eq. 3), solved exactly here
    w = 2 * np.pi * f
    tau = -2 * a0 * c0 ** (nu - 1)
    eta = 2 * a0 * c0 ** nu * np.tan(np.pi * nu / 2)
    K = complex(k0)
    for _ in range(200):
        K = np.sqrt(k0 ** 2 - 1j * tau * w * K ** nu + eta * K ** (nu + 1))
    alpha = a0 * w ** nu
    assert abs(K - (k0 + alpha * (np.tan(np.pi * nu / 2) + 1j))) < 0.1 * alpha      # the first-order form
    ratio = abs(res.p[0, b]) / abs(res.p[0, a])
    assert abs(ratio / np.exp(-K.imag * (b - a) * dx) - 1) < 0.01, ratio
    dphi = np.unwrap(np.angle(res.p[0, a:b + 1]))
    Kre = (dphi[-1] - dphi[0]) / ((b - a) * dx)
    assert abs(Kre / K.real - 1) < 1e-3


def test_kspace_potential_plus_scatterer_reduces_to_both_parents_and_to_the_typed_formula():
    """solve_kspace(..., Us): (i) Us = 0 is Eq. 24 alone; (ii) a lossless multiplier VV = -i eps makes it the
    ordinary series with V = U_s - i eps (Eq. 26); (iii) against the iteration typed with numpy's
    FFT on the periodic grid: psi <- A ifft2(g (VV fft2(psi) + fft2(U_s psi + S)))  (Eq. 24 + the U_s term of Eq. 25)."""
    N, dx, f, c0 = 32, 1.0e-4, 1.0e6, 1500.0
    k0, eps = R.wavenumber(f, c0, 0.8)
    S = np.zeros((N, N), dtype=np.complex128)
    S[10:22, 6] = -1.0e6j
    yy, xx = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    Us = np.where((xx - 20) ** 2 + (yy - 15) ** 2 <= 16, (2 * np.pi * f / 1650.0) ** 2 - k0 * k0, 0.0).astype(np.complex128)
    g = R.green_spectrum((N, N), dx, k0, eps)
    VV = R.kspace_potential((N, N), dx, 5.5e-10 * 50, 1.5, f, c0, 0.8)
    win = tuple(R.abl_window(N, 6) for _ in range(2))
    A = np.outer(win[1], win[0])
    # (i)
    a = R.solve_kspace(S, g, VV, 25, 0.0, pad=1, windows=win)
    b = R.solve_kspace(S, g, VV, 25, 0.0, pad=1, windows=win, Us=np.zeros_like(Us))
    assert np.allclose(a.p, b.p, rtol=0, atol=1e-13 * np.abs(a.p).max()) and np.allclose(a.history, b.history)
    # (ii)
    lossless = np.full((N, N), -1j * eps)
    c_ = R.solve_kspace(S, g, lossless, 25, 0.0, pad=1, windows=win, Us=Us)
    d = R.solve(Us - 1j * eps, S, g, 25, 0.0, pad=1, windows=win)
    assert np.allclose(c_.p, d.p, rtol=0, atol=1e-12 * np.abs(d.p).max()) and np.allclose(c_.history, d.history, rtol=1e-10)
    # (iii) the Picard iterates typed out
    res = R.solve_kspace(S, g, VV, 12, 0.0, pad=1, windows=win, Us=Us)
    u = A * np.fft.ifft2(g * np.fft.fft2(S))
    p = u.copy()
    for _ in range(12):
        u = A * np.fft.ifft2(g * (VV * np.fft.fft2(u) + np.fft.fft2(Us * u)))
        p += u
    assert np.abs(res.p - p).max() <= 1e-12 * np.abs(p).max()
    # and the scatterer does change the field (the pin is not vacuous)
    assert np.abs(res.p - R.solve_kspace(S, g, VV, 12, 0.0, pad=1, windows=win).p).max() > 1e-3 * np.abs(p).max()
