"""Pins P6 (dense Lippmann-Schwinger solve) and P7 (invariants) of the CPU oracle.  CPU only."""
import numpy as np
import pytest

import oracle.tbs_ref as R


def _small_problem(N, seed, ndim=2, contrast=1.0):
    """Disc/ball scatterer + 1 % noise + absorption on an N^d grid at 6 points per wavelength."""
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / 6.0
    rng = np.random.default_rng(seed)
    shape = (N,) * ndim
    ax = np.arange(N) - (N - 1) / 2
    grids = np.meshgrid(*([ax] * ndim), indexing="ij")
    r = np.sqrt(sum(g ** 2 for g in grids))
    c = np.full(shape, c0) * (1.0 + 0.01 * rng.standard_normal(shape))
    c[r < N / 5] *= 1.0 + 0.08 * contrast
    V = R.potential(c, 0.75, 1.5, f, c0, 0.8)
    k0, eps = R.wavenumber(f, c0, 0.8)
    g = R.green_spectrum(tuple(2 * s for s in shape), dx, k0, eps)
    S = np.zeros(shape, complex)
    S[(1,) * ndim] = 1.0
    S[(2,) + (N // 2,) * (ndim - 1)] = 0.5j
    return dx, V, S, g


def _dense_G(g, shape):
    """G[a, b] = g_disc[(a - b) mod M] with g_disc = IDFT_M(ghat) (numpy's ifftn: library routine)."""
    gd = np.fft.ifftn(g)
    n = int(np.prod(shape))
    idx = np.array(list(np.ndindex(*shape)))
    M = np.array(g.shape)
    G = np.empty((n, n), complex)
    for a in range(n):
        d = (idx[a][None, :] - idx) % M[None, :]
        G[a, :] = gd[tuple(d.T)]
    return G


@pytest.mark.parametrize("N", [16, 24])
def test_series_limit_equals_dense_direct_solve(N):
    """Eq. 17: psi = G V psi + G S  <=>  (I - G diag V) p = G S."""
    dx, V, S, g = _small_problem(N, N)
    G = _dense_G(g, (N, N))
    n = N * N
    A = np.eye(n) - G * V.reshape(1, n)
    p_dense = np.linalg.solve(A, G @ S.reshape(n)).reshape(N, N)
    res = R.solve(V, S, g, 5000, 1e-13)
    assert res.status == R.OK
    err = np.linalg.norm(res.p - p_dense) / np.linalg.norm(p_dense)
    assert err < 1e-10
    # G is symmetric (convolution with an even kernel)
    assert np.abs(G - G.T).max() < 1e-13 * np.abs(G).max()
    # geometric tail: ||u_{n+1}||/||u_n|| -> spectral radius of G diag V, which is < 1
    rho = np.abs(np.linalg.eigvals(G * V.reshape(1, n))).max()
    assert rho < 1.0
    h = res.history
    k = res.n_terms
    pn = np.linalg.norm(res.p)
    tail = (h[k] * pn) / (h[k - 1] * pn)          # p is converged, so ||p_n|| is constant here
    assert abs(tail - rho) < 1e-2 and tail < 1.0


def test_series_limit_equals_dense_direct_solve_3d():
    N = 6
    dx, V, S, g = _small_problem(N, 3, ndim=3)
    G = _dense_G(g, (N,) * 3)
    n = N ** 3
    A = np.eye(n) - G * V.reshape(1, n)
    p_dense = np.linalg.solve(A, G @ S.reshape(n)).reshape((N,) * 3)
    res = R.solve(V, S, g, 5000, 1e-13)
    assert res.status == R.OK
    assert np.linalg.norm(res.p - p_dense) / np.linalg.norm(p_dense) < 1e-10


def test_dense_limit_with_abl_window():
    """With a window the limit is p = (I - A G diag V)^-1 A G S."""
    N = 16
    dx, V, S, g = _small_problem(N, 5)
    a = R.abl_window(N, 4)
    G = _dense_G(g, (N, N))
    n = N * N
    Aw = np.outer(a, a).reshape(n, 1)
    p_dense = np.linalg.solve(np.eye(n) - Aw * G * V.reshape(1, n), Aw[:, 0] * (G @ S.reshape(n)))
    res = R.solve(V, S, g, 5000, 1e-13, windows=(a, a))
    assert np.linalg.norm(res.p.reshape(n) - p_dense) / np.linalg.norm(p_dense) < 1e-10


# ---------------------------------------------------------------- P7 invariants
def test_reciprocity():
    """R = (I - G V)^-1 G is symmetric: field at b from a unit source at a equals field at a
    from a unit source at b, for any V (A == 1)."""
    N = 24
    dx, V, _, g = _small_problem(N, 11)
    a, b = (3, 5), (17, 12)
    Sa = np.zeros((N, N), complex)
    Sb = np.zeros((N, N), complex)
    Sa[a] = 1.0
    Sb[b] = 1.0
    pa = R.solve(V, Sa, g, 5000, 1e-13).p
    pb = R.solve(V, Sb, g, 5000, 1e-13).p
    assert abs(pa[b] - pb[a]) < 1e-11 * abs(pa[b])


def test_zero_potential_gives_zero_corrections():
    N = 16
    dx, V, S, g = _small_problem(N, 2)
    res = R.solve(np.zeros_like(V), S, g, 10, 1e-6)
    assert res.n_terms == 1 and res.history[1] == 0.0 and res.status == R.OK
    assert np.array_equal(res.p, R.apply_G(S, g))
    assert np.all(res.u_last == 0)


def test_superposition_and_mirror_symmetry():
    N = 16
    dx, V, S, g = _small_problem(N, 7)
    S2 = np.roll(S, (3, 2), (0, 1))
    nt = 12
    p1 = R.solve(V, S, g, nt, 0.0).p
    p2 = R.solve(V, S2, g, nt, 0.0).p
    p12 = R.solve(V, 2.0 * S - 1j * S2, g, nt, 0.0).p
    assert np.allclose(p12, 2.0 * p1 - 1j * p2, rtol=1e-12, atol=1e-14 * np.abs(p12).max())
    # mirror i -> N-1-i along x
    pm = R.solve(V[:, ::-1], S[:, ::-1], g, nt, 0.0).p
    assert np.allclose(pm[:, ::-1], p1, rtol=1e-11, atol=1e-13 * np.abs(p1).max())
    # transpose x <-> y
    pt = R.solve(V.T.copy(), S.T.copy(), g, nt, 0.0).p
    assert np.allclose(pt.T, p1, rtol=1e-11, atol=1e-13 * np.abs(p1).max())


def test_term_form_equals_picard_form():
    """Eq. 18 vs Eq. 19: sum_{m<=l} u_m = psi^l with psi^0 = G S,
    psi^{l+1} = G(V psi^l + S) -- the paper's own iteration, written with apply_G."""
    N = 16
    dx, V, S, g = _small_problem(N, 9)
    psi = R.apply_G(S, g)
    for l in range(1, 9):
        psi = R.apply_G(V * psi + S, g)
        res = R.solve(V, S, g, l, 0.0)
        assert res.n_terms == l
        assert np.allclose(res.p, psi, rtol=1e-12, atol=1e-14 * np.abs(psi).max())
        # history is ||u_l|| / ||p_l|| with u_l = p_l - p_{l-1}
    prev = R.solve(V, S, g, 7, 0.0).p
    last = R.solve(V, S, g, 8, 0.0)
    assert abs(last.history[8] - np.linalg.norm(last.p - prev) / np.linalg.norm(last.p)) < 1e-9
    assert np.allclose(last.u_last, last.p - prev, atol=1e-12 * np.abs(last.p).max())


def test_stops_at_first_term_below_tol_and_reports_not_converged():
    N = 16
    dx, V, S, g = _small_problem(N, 13)
    full = R.solve(V, S, g, 400, 0.0)
    tol = 1e-4
    k = int(np.argmax(full.history[1:] < tol)) + 1
    res = R.solve(V, S, g, 400, tol)
    assert res.status == R.OK and res.n_terms == k
    assert np.array_equal(res.history, full.history[:k + 1])
    capped = R.solve(V, S, g, k - 1, tol)
    assert capped.status == R.NOT_CONVERGED and capped.n_terms == k - 1


def test_divergence_is_reported():
    """||G V|| > 1: a strong extended potential makes the series blow up."""
    N = 16
    dx, V, S, g = _small_problem(N, 1)
    res = R.solve(40.0 * V.real + 0j, S, g, 4000, 1e-12)
    assert res.status in (R.ERR_DIVERGED, R.NOT_CONVERGED)
    assert res.history[res.n_terms] > 1e-12 or not np.isfinite(res.history[res.n_terms])
