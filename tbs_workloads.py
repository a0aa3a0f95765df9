"""Seeded synthetic inputs shaped like the paper's workloads (DESIGN.md
"Input recipe").  Serves BOTH the CUDA path and the oracle and therefore holds none of the
method's arithmetic: it only draws media (sound speed / density maps), element positions and
element amplitudes.  The paper's workloads are themselves synthetic (a line source in analytic
media); no public dataset is involved.

Axis convention: arrays are numpy (z, y, x) / (y, x) with x fastest; the array lies along x at
row ``y_src`` (2D) / plane ``z_src`` (3D).  Positions are metres, cell (0,0,0) centre at r = 0,
columns ordered (x, y[, z]).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED0 = 20250713


@dataclass
class Workload:
    name: str
    ndim: int
    shape: tuple            # numpy shape, (y, x) or (z, y, x)
    dx: float
    freqs: list             # Hz
    c0: float
    rho0: float
    damping: float
    alpha0_db: float        # dB / (MHz^y cm)
    y: float
    beta: float
    c: np.ndarray           # float32 sound-speed map, m/s
    rho: np.ndarray | None  # float32 density map (does not enter V, reading A7)
    src_pos: np.ndarray     # float64 [n_src][ndim]  (x, y[, z]) metres
    src_amp: np.ndarray     # complex64 [nfreq][n_src]
    tol: float
    max_terms: int
    notes: dict = field(default_factory=dict)

    @property
    def n_points(self) -> int:
        return int(np.prod(self.shape))


def _grf(rng, shape, dx, corr_len_m):
    """White N(0,1) noise periodically convolved with exp(-r^2/(2 l^2)), min-max scaled to [0,1]."""
    g = rng.standard_normal(shape).astype(np.float64)
    G = np.fft.rfftn(g)
    for ax, n in enumerate(shape):
        k = np.fft.rfftfreq(n) if ax == len(shape) - 1 else np.fft.fftfreq(n)
        # FT of a Gaussian of std l (in cells) is a Gaussian exp(-2 pi^2 l^2 k^2)
        l_cells = corr_len_m / dx
        w = np.exp(-2.0 * (math.pi * l_cells * k) ** 2)
        sh = [1] * len(shape)
        sh[ax] = w.size
        G *= w.reshape(sh)
    g = np.fft.irfftn(G, s=shape, axes=tuple(range(len(shape))))
    g -= g.min()
    g /= g.max()
    return g


def _linear_array_x(n_el, pitch, nx, dx):
    """x positions of n_el elements of given pitch, centred on the grid."""
    xc = 0.5 * (nx - 1) * dx
    return xc + (np.arange(n_el) - 0.5 * (n_el - 1)) * pitch


def _fit_elements(n_el, pitch, nx, dx):
    """Shrink the element count (keeping the pitch) so the array spans <= 60 % of the width."""
    width = (nx - 1) * dx
    while n_el > 2 and (n_el - 1) * pitch > 0.6 * width:
        n_el //= 2
    return n_el


def cfg1(N: int = 128) -> Workload:
    """2D homogeneous lossless, 16 in-phase point elements at row 8 (shape of paper E1)."""
    dx, f, c0 = 0.25e-3, 1.0e6, 1500.0
    cols = np.arange(N // 2 - 8, N // 2 + 8)
    pos = np.stack([cols * dx, np.full(cols.size, 8 * dx)], axis=1)
    amp = np.ones((1, cols.size), dtype=np.complex64)
    return Workload("cfg1_2d_%d_lossless" % N, 2, (N, N), dx, [f], c0, 1000.0, 0.8, 0.0, 1.5, 1.0,
                    np.full((N, N), c0, dtype=np.float32), None, pos, amp, 1e-7, 2000)


def cfg2(N: int = 1024) -> Workload:
    """2D homogeneous absorbing/dispersive, focused Hann-apodised 64-element array (paper E2)."""
    f, c0 = 2.5e6, 1540.0
    dx = c0 / f / 6.0
    n_el = _fit_elements(64, 0.3e-3, N, dx)
    x = _linear_array_x(n_el, 0.3e-3, N, dx)
    pos = np.stack([x, np.full(n_el, 16 * dx)], axis=1)
    j = np.arange(n_el)
    hann = 0.5 * (1.0 - np.cos(2.0 * math.pi * (j + 1) / (n_el + 1)))
    F = 30e-3
    xr = x - x.mean()
    k0 = 2.0 * math.pi * f / c0
    amp = (hann * np.exp(-1j * k0 * (np.sqrt(xr ** 2 + F ** 2) - F))).astype(np.complex64)[None, :]
    return Workload("cfg2_2d_%d_absorbing" % N, 2, (N, N), dx, [f], c0, 1000.0, 0.8, 0.75, 1.5, 1.0,
                    np.full((N, N), c0, dtype=np.float32), np.full((N, N), 1000.0, dtype=np.float32),
                    pos, amp, 1e-6, 4000)


def cfg3(N: int = 2048, seed: int = SEED0 + 3) -> Workload:
    """2D inhomogeneous: Gaussian random c in [1450,1600] + 5 discs (+-3 %), absorbing (paper E3 extended)."""
    f, c0 = 2.0e6, 1525.0
    dx = c0 / f / 6.0
    rng = np.random.default_rng(seed)
    c = 1450.0 + 150.0 * _grf(rng, (N, N), dx, 2e-3)
    rho = 950.0 + 150.0 * _grf(rng, (N, N), dx, 2e-3)
    L = (N - 1) * dx
    yy, xx = np.meshgrid(np.arange(N) * dx, np.arange(N) * dx, indexing="ij")
    margin = min(8e-3, 0.2 * L)
    discs = []
    for _ in range(5):
        r = rng.uniform(1e-3, 4e-3) * min(1.0, N / 2048.0 * 4.0)
        cx = rng.uniform(margin, L - margin)
        cy = rng.uniform(margin + 16 * dx, L - margin)
        sgn = 1.0 if rng.random() < 0.5 else -1.0
        m = (xx - cx) ** 2 + (yy - cy) ** 2 <= r * r
        c[m] *= 1.0 + 0.03 * sgn
        discs.append((cx, cy, r, sgn))
    n_el = _fit_elements(128, 0.2e-3, N, dx)
    x = _linear_array_x(n_el, 0.2e-3, N, dx)
    pos = np.stack([x, np.full(n_el, 16 * dx)], axis=1)
    amp = np.ones((1, n_el), dtype=np.complex64)
    return Workload("cfg3_2d_%d_inhomogeneous" % N, 2, (N, N), dx, [f], c0, 1025.0, 0.8, 0.5, 1.1, 1.0,
                    c.astype(np.float32), rho.astype(np.float32), pos, amp, 1e-6, 6000,
                    notes={"discs": discs})


def cfg4(N: int = 4096) -> Workload:
    """2D nonlinear homogeneous tissue: fundamental 1.5 MHz, then 3 MHz driven by p1^2 (paper E4)."""
    f1, c0 = 1.5e6, 1540.0
    dx = c0 / (2.0 * f1) / 8.0
    n_el = _fit_elements(128, 0.3e-3, N, dx)
    x = _linear_array_x(n_el, 0.3e-3, N, dx)
    pos = np.stack([x, np.full(n_el, 16 * dx)], axis=1)
    amp = np.ones((1, n_el), dtype=np.complex64)
    return Workload("cfg4_2d_%d_nonlinear" % N, 2, (N, N), dx, [f1], c0, 1050.0, 0.8, 0.6, 1.2, 4.5,
                    np.full((N, N), c0, dtype=np.float32), None, pos, amp, 1e-6, 8000,
                    notes={"surface_pressure_pa": 1.0e6})


def cfg5(N: int = 256, nfreq: int = 1, seed: int = SEED0 + 5) -> Workload:
    """3D inhomogeneous medium, 64 rectangular elements each sampled by 4x32 points (paper has no 3D).

    nfreq = 1: f = 1 MHz; nfreq = 16: the broadband batch f_i = 0.5 + 0.1 i MHz."""
    c0 = 1525.0
    dx = c0 / 1.0e6 / 6.0
    freqs = [1.0e6] if nfreq == 1 else [0.5e6 + 0.1e6 * i for i in range(nfreq)]
    rng = np.random.default_rng(seed)
    c = 1450.0 + 150.0 * _grf(rng, (N, N, N), dx, 2e-3)
    rho = 950.0 + 150.0 * _grf(rng, (N, N, N), dx, 2e-3)
    n_el = _fit_elements(64, 0.25e-3, N, dx)
    xe = _linear_array_x(n_el, 0.25e-3, N, dx)
    yc = 0.5 * (N - 1) * dx
    w_el = 0.2e-3
    h_el = min(4e-3, 0.5 * (N - 1) * dx)
    a = ((np.arange(4) + 0.5) / 4.0 - 0.5) * w_el
    b = ((np.arange(32) + 0.5) / 32.0 - 0.5) * h_el
    px = (xe[:, None, None] + a[None, :, None] + 0 * b[None, None, :]).reshape(-1)
    py = (yc + 0 * xe[:, None, None] + 0 * a[None, :, None] + b[None, None, :]).reshape(-1)
    pz = np.full(px.size, 8 * dx)
    pos = np.stack([px, py, pz], axis=1)
    amp = np.full((len(freqs), px.size), 1.0 / 128.0, dtype=np.complex64)
    return Workload("cfg5_3d_%d_inhomogeneous_f%d" % (N, len(freqs)), 3, (N, N, N), dx, freqs, c0,
                    1025.0, 0.8, 0.5, 1.1, 1.0, c.astype(np.float32), rho.astype(np.float32),
                    pos, amp, 1e-6, 6000)


CONFIGS = {1: cfg1, 2: cfg2, 3: cfg3, 4: cfg4, 5: cfg5}


def paper_e1(N: int = 4096) -> Workload:
    """The paper's own first experiment: N = 4096, dx = 0.02 mm, homogeneous lossless water,
    f = the 55th harmonic of the periodic grid, 501-pixel line source of strength -i 10^6 along y at column
    675, centred on row 2049 (1-based).  notes carries the paper-faithful solver options: periodic boundary,
    450-cell layer with zeta mu/2 = 9.666, Eq. 30 on the centre row below 10^-5, cap 2000 iterations.  Smaller
    N keep dx, the frequency, and scale the geometry."""
    dx, c0 = 0.02e-3, 1500.0
    f = 55 * c0 / (4096 * dx)
    k = N / 4096.0
    row = N // 2
    half = int(round(250 * k))
    rows = np.arange(row - half, row + half + 1)
    pos = np.stack([np.full(rows.size, round(675 * k) * dx), rows * dx], 1).astype(np.float64)
    amp = np.full((1, rows.size), -1.0e6j, dtype=np.complex64)
    return Workload(name=f"paper_e1_2d_{N}_periodic", ndim=2, shape=(N, N), dx=dx, freqs=[f], c0=c0, rho0=1000.0,
                    damping=0.8, alpha0_db=0.0, y=1.5, beta=3.5, c=np.full((N, N), c0, dtype=np.float32), rho=None,
                    src_pos=pos, src_amp=amp, tol=1e-5, max_terms=2000,
                    notes={"boundary": "periodic", "abl_cells": int(round(450 * k)), "zeta_half_mu": 9.666,
                           "criterion_row": row})


def make(idx: int, **kw) -> Workload:
    return CONFIGS[idx](**kw)
