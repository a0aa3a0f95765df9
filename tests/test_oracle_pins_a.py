"""Pins P1, P8 and the small setup functions of the CPU oracle.

Each test checks oracle/ against something other than itself: numbers the paper prints
(tests/golden/paper_constants.txt), a library routine (numpy.fft), a naive DFT matrix, or an
independent numerical derivation.  CPU only.
"""
import math

import numpy as np
import pytest

import oracle.tbs_ref as R


# ---------------------------------------------------------------- P8: hand-written FFT
@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 32, 64, 24, 48, 12])
@pytest.mark.parametrize("sign", [-1, 1])
def test_fft_vs_naive_dft_matrix(n, sign):
    rng = np.random.default_rng(n * 7 + sign)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    j = np.arange(n)
    F = np.exp(sign * 2j * np.pi * np.outer(j, j) / n)
    assert np.allclose(R.fft1d(x, sign), F @ x, rtol=0, atol=1e-12 * n)


@pytest.mark.parametrize("n", [256, 1024, 4096])
def test_fft_vs_numpy_and_roundtrip(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = R.fft1d(x, -1)
    assert np.abs(X - np.fft.fft(x)).max() < 1e-11 * math.sqrt(n)
    # Parseval and round trip
    assert abs(np.vdot(X, X).real / n - np.vdot(x, x).real) < 1e-10 * n
    assert np.abs(R.fft1d(X, +1) / n - x).max() < 1e-13 * math.log2(n) * 4


def test_fft_impulse_and_constant():
    n = 64
    e = np.zeros(n, complex)
    e[3] = 1.0
    k = np.arange(n)
    assert np.allclose(R.fft1d(e, -1), np.exp(-2j * np.pi * 3 * k / n), atol=1e-14)
    c = np.ones(n, complex)
    X = R.fft1d(c, -1)
    assert abs(X[0] - n) < 1e-12 and np.abs(X[1:]).max() < 1e-12


# ---------------------------------------------------------------- P1: printed constants
def test_frequency_and_wavenumber_printed(golden):
    f = golden["f_multiple"] * golden["v_f"] / (golden["n_grid"] * golden["dx_m"])
    assert abs(f - golden["f_hz"]) < 0.5            # PAPER.md:251 prints 1007080
    k0, eps = R.wavenumber(golden["f_hz"], golden["v_f"], golden["eps_over_k2"])
    assert abs(k0 * golden["a_m"] - golden["kf_a"]) < 0.005   # k_f a = 4.22
    assert abs(eps / k0 ** 2 - 0.8) < 1e-15


def test_potential_lossless_is_alg1_case3(golden):
    """Alg. 1 l.23-29: V = (k_s^2 - k_f^2, -eps) inside, (0, -eps) outside."""
    f, vf = golden["f_hz"], golden["v_f"]
    c = np.array([vf, 1350.0, 1650.0, 1800.0])
    V = R.potential(c, 0.0, 1.5, f, vf, 0.8)
    w = 2 * math.pi * f
    kf = w / vf
    expect = (w / c) ** 2 - kf ** 2 - 1j * 0.8 * kf ** 2
    assert np.allclose(V, expect, rtol=1e-13)
    assert V[0].real == 0.0 or abs(V[0].real) < 1e-6


def test_potential_absorbing_matches_eq24_on_shell(golden):
    """Reading A6: on-shell (|p| = k_f) the paper's k-space multiplier of Eq. 24,
    -i tau w k^nu + eta k^(nu+1) - i eps with tau, eta of PAPER.md:58, equals the spatial
    potential ktilde^2 - k_f^2 - i eps to first order in alpha/k.  tau and eta are also the
    values Table 4 prints."""
    f, vf, nu, a0 = golden["f_hz"], golden["v_f"], golden["nu"], golden["alpha0_si"]
    tau = -2 * a0 * vf ** (nu - 1)
    eta = 2 * a0 * vf ** nu * math.tan(math.pi * nu / 2)
    assert abs(tau - golden["tau"]) < 0.05e-8          # prints -4.3e-8
    assert abs(eta - golden["eta"]) < 0.05e-5          # prints -6.4e-5
    w = 2 * math.pi * f
    kf = w / vf
    eps = 0.8 * kf ** 2
    VV = -1j * tau * w * kf ** nu + eta * kf ** (nu + 1) - 1j * eps
    a0_db = a0 * 8.685889638 * (2 * math.pi * 1e6) ** nu / 100.0   # Np(rad/s)^-nu/m -> dB/(MHz^nu cm)
    assert abs(a0_db - 0.752) < 1e-3
    V = R.potential(np.array([vf]), a0_db, nu, f, vf, 0.8)[0]
    alpha = a0 * w ** nu
    # difference is the alpha^2 term: |alpha (tan + i)|^2
    assert abs(V - VV) <= 2.1 * alpha ** 2
    assert abs(V - VV) / abs(VV + 1j * eps) < 2 * alpha / kf      # first order in alpha/k
    # Im ktilde = alpha (Eq. 3): sqrt(V + k_f^2 + i eps) has imaginary part alpha
    kt = np.sqrt(V + kf ** 2 + 1j * eps)
    assert abs(kt.imag - alpha) < 1e-9 * alpha + 1e-12


def test_potential_alpha_map_equals_scalar():
    c = np.linspace(1450, 1600, 7)
    a = R.potential(c, 0.5, 1.1, 2e6, 1525.0, 0.8)
    b = R.potential(c, np.full(7, 0.5), 1.1, 2e6, 1525.0, 0.8)
    assert np.array_equal(a, b)


# ---------------------------------------------------------------- ABL, Eq. 29
def test_abl_window_matches_eq29_in_paper_units(golden):
    n, cells = int(golden["n_grid"]), int(golden["abl_cells"])
    zeta, dx_cm = golden["zeta_np_per_cm"], golden["dx_m"] * 100.0
    mu = cells * dx_cm
    a = R.abl_window(n, cells, zeta * mu / 2)
    i = np.arange(cells)
    expect = 1.0 / (1.0 + np.exp(-zeta * (i * dx_cm - 0.5 * mu)))     # PAPER.md:253 Eq. 29
    assert np.allclose(a[:cells], expect, rtol=1e-12)
    assert np.allclose(a[::-1], a)                      # all faces alike
    assert np.all(a[cells:n - cells] == 1.0)
    assert np.all(np.diff(a[:cells]) > 0)
    assert abs(zeta * mu / 2 - 9.666) < 1e-3


def test_abl_zero_cells_is_identity():
    assert np.all(R.abl_window(32, 0) == 1.0)


# ---------------------------------------------------------------- source deposition (A9)
def test_deposit_on_node_is_single_pixel(golden):
    """Alg. 1 l.14-18: S = (0, -1e6) at the element pixel, 0 elsewhere."""
    dx = golden["dx_m"]
    S = R.deposit((16, 16), dx, [[5 * dx, 9 * dx]], [-1j * golden["source_strength"]])
    assert S[9, 5] == -1e6j
    S[9, 5] = 0
    assert np.all(S == 0)


@pytest.mark.parametrize("nd", [1, 2, 3])
def test_deposit_weights_conserve_mass_and_first_moment(nd):
    rng = np.random.default_rng(nd)
    shape = (9, 8, 7)[-nd:]
    dx = 0.3e-3
    n_src = 11
    pos = np.stack([rng.uniform(0, (shape[nd - 1 - a] - 1) * dx, n_src) for a in range(nd)], 1)
    amp = rng.standard_normal(n_src) + 1j * rng.standard_normal(n_src)
    S = R.deposit(shape, dx, pos, amp)
    assert abs(S.sum() - amp.sum()) < 1e-12
    grids = np.meshgrid(*[np.arange(s) * dx for s in shape], indexing="ij")
    for a in range(nd):
        coord = grids[nd - 1 - a]
        assert abs((S * coord).sum() - (amp * pos[:, a]).sum()) < 1e-14


def test_deposit_rejects_outside():
    with pytest.raises(ValueError):
        R.deposit((8, 8), 1e-3, [[9e-3, 1e-3]], [1.0])


# ---------------------------------------------------------------- second-harmonic source
def test_second_harmonic_source_is_2w_component_of_westervelt(golden):
    """Eq. 11 with Psi = Re(psi1 e^{-iwt}): the e^{-2iwt} component of
    xi d^2(Psi^2)/dt^2 moved to the right-hand side is -S2 = xi (2w)^2 psi1^2/2 (Eq. 27b,
    PAPER.md:217), i.e. S2 = -xi (2w)^2 psi1^2 / 2 (Eq. 28b).  Checked by a
    numerical time derivative and projection, not by retyping the formula."""
    f = golden["f_hz"]
    w = 2 * math.pi * f
    beta = 1 + golden["b_over_a"] / 2
    rho, c = golden["rho_f"], golden["v_f"]
    xi = beta / (rho * c ** 4)
    psi1 = np.array([0.7 - 1.3j, 2.0 + 0.5j]) * 1e5
    S2 = R.second_harmonic_source(psi1, beta, rho, c, f)
    nt = 4096
    t = np.arange(nt) / nt * (2 * math.pi / w)           # one fundamental period
    dt = t[1] - t[0]
    for i, a in enumerate(psi1):
        Psi2 = (a * np.exp(-1j * w * t)).real ** 2
        d2 = (np.roll(Psi2, -1) - 2 * Psi2 + np.roll(Psi2, 1)) / dt ** 2      # periodic FD
        # component multiplying e^{-2iwt}:  X(t) = Re(x e^{-2iwt}) -> x = 2 <X e^{+2iwt}>
        comp = 2 * np.mean(xi * d2 * np.exp(2j * w * t))
        # equation: lap psi2 + k2^2 psi2 + comp = 0  ->  rhs = -comp = -S2
        assert abs(S2[i] - comp) < 2e-5 * abs(comp)


@pytest.mark.parametrize("h", [2, 3, 4, 5])
def test_harmonic_sources_are_sum_frequency_components_of_westervelt(golden, h):
    """Eqs. 27b-27e / 28b-28e: with Psi = Re(Psi+), Psi+ = sum_m psi_m e^{-i m w t},
    Psi^2 = (Psi+^2 + Psi+*^2)/4 + |Psi+|^2/2; the paper keeps the sum-frequency part Re(Psi+^2)/2 and
    drops the difference terms.  S_h is minus the e^{-i h w t} component of
    xi d^2/dt^2 of that part -- evaluated here by a numerical time derivative and projection."""
    f = golden["f_hz"]
    w = 2 * math.pi * f
    beta = 1 + golden["b_over_a"] / 2
    rho, c = golden["rho_f"], golden["v_f"]
    xi = beta / (rho * c ** 4)
    rng = np.random.default_rng(5)
    psi = [(rng.standard_normal(3) + 1j * rng.standard_normal(3)) * s for s in (1e5, 3e4, 1e4, 3e3)]
    S = R.harmonic_source(h, psi, beta, rho, c, f)
    nt = 8192
    t = np.arange(nt) / nt * (2 * math.pi / w)
    dt = t[1] - t[0]
    for i in range(3):
        plus = sum(psi[m][i] * np.exp(-1j * (m + 1) * w * t) for m in range(h - 1))
        X = (plus ** 2).real / 2
        d2 = (np.roll(X, -1) - 2 * X + np.roll(X, 1)) / dt ** 2
        comp = 2 * np.mean(xi * d2 * np.exp(1j * h * w * t))
        assert abs(S[i] - comp) < 1e-4 * abs(comp)
    if h == 2:
        assert np.allclose(S, R.second_harmonic_source(psi[0], beta, rho, c, f), rtol=1e-14)
