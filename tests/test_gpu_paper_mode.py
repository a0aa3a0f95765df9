"""GPU parity of the paper-faithful options: periodic N-grid FFTs, the absorbing layer
on the whole field, the centre-row L1 criterion of Eq. 30; and the paper's homogeneous case itself."""
import numpy as np
import pytest
import torch

import oracle.tbs_ref as R
from parity_util import compare_fields, compare_history

pytestmark = pytest.mark.gpu


def _case(N, abl):
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / 6.0
    rng = np.random.default_rng(N)
    c = (c0 * (1 + 0.01 * rng.standard_normal((N, N)))).astype(np.float32)
    yy, xx = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    c[(xx - 0.6 * N) ** 2 + (yy - 0.5 * N) ** 2 < (N / 10) ** 2] = 1580.0
    rows = np.arange(N // 2 - N // 8, N // 2 + N // 8 + 1)
    pos = np.stack([np.full(rows.size, (abl + 6) * dx), rows * dx], 1)
    amp = np.full((1, rows.size), -1.0e6j, dtype=np.complex64)
    return f, c0, dx, c, pos, amp


def _plan(N, abl, f, c0, dx, c, pos, amp):
    from paper_2507_13754_b200.tbs import Plan
    plan = Plan((N, N), dx, [f], c0, 0.8)
    plan.set_boundary("periodic")
    plan.set_abl(abl, 9.666)
    plan.set_medium(torch.from_numpy(c).cuda(), alpha0_db=0.5, y=1.1)
    plan.set_source(pos, amp)
    return plan


def _oracle_inputs(N, abl, f, c0, dx, c, pos, amp):
    k0, eps = R.wavenumber(f, c0, 0.8)
    V = R.potential(c.astype(np.float64), 0.5, 1.1, f, c0, 0.8)
    S = R.deposit((N, N), dx, pos, amp[0])
    g = R.green_spectrum((N, N), dx, k0, eps)          # the N-grid itself: pad factor 1
    win = tuple(R.abl_window(N, abl) for _ in range(2))
    return V, S, g, win


def test_periodic_boundary_matches_oracle_pad_factor_one():
    N, abl = 128, 16
    case = _case(N, abl)
    V, S, g, win = _oracle_inputs(N, abl, *case)
    ref = R.solve(V, S, g, 3000, 1e-6, pad=1, windows=win)
    res = _plan(N, abl, *case).solve(3000, 1e-6)
    assert res.status == 0 and ref.status == R.OK
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, "periodic 128^2")


@pytest.mark.parametrize("shape", [(32, 32), (64, 128), (128, 64), (256, 256), (512, 1024), (1024, 32), (32, 1024),
                                   (2048, 64), (64, 2048), (4096, 32), (32, 4096), (2048, 2048)])
def test_unpadded_periodic_kernels_apply_green_every_length(shape):
    """The unpadded kernels (k_row / k_conv <..., PER>: two lines per packed value) at every transform length in
    both axes: one application of G on the periodic N-grid against the oracle's pad-factor-1 definition."""
    from paper_2507_13754_b200.tbs import Plan
    rng = np.random.default_rng(sum(shape) + 1)
    x = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
    dx = 1500.0 / 1.0e6 / 6.0
    plan = Plan(shape, dx, [1.0e6], 1500.0, 0.8)
    plan.set_boundary("periodic")
    out = plan.apply_green(0, torch.from_numpy(x).cuda()).cpu().numpy()
    k0, eps = R.wavenumber(1.0e6, 1500.0, 0.8)
    ref = R.apply_G(x.astype(np.complex128), R.green_spectrum(shape, dx, k0, eps), 1)
    rel = np.linalg.norm(out - ref) / np.linalg.norm(ref)
    assert rel < 2e-6, rel
    # switching back to the padded boundary on the same plan restores the linear convolution
    plan.set_boundary("pad")
    if max(shape) <= 1024:
        out2 = plan.apply_green(0, torch.from_numpy(x).cuda()).cpu().numpy()
        ref2 = R.apply_G(x.astype(np.complex128), R.green_spectrum(tuple(2 * s for s in shape), dx, k0, eps))
        assert np.linalg.norm(out2 - ref2) / np.linalg.norm(ref2) < 2e-6


def test_periodic_boundary_512_matches_oracle_pad_factor_one():
    """N = 512, 40 terms with the absorbing layer, history term by term."""
    N, abl = 512, 32
    case = _case(N, abl)
    V, S, g, win = _oracle_inputs(N, abl, *case)
    ref = R.solve(V, S, g, 40, 0.0, pad=1, windows=win)
    res = _plan(N, abl, *case).solve(40, 0.0)
    assert int(res.n_terms[0]) == ref.n_terms == 40
    compare_fields(res.p[0].cpu().numpy(), ref.p, "periodic 512^2, 40 terms")
    compare_history(res.history[0], ref.history, 40)


def test_periodic_boundary_3d_matches_oracle_pad_factor_one():
    """3-D: in the z pass whole tiles sit at a masked ky and the state of a line changes from tile to tile."""
    from paper_2507_13754_b200.tbs import Plan
    N, abl = 32, 6
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / 6.0
    rng = np.random.default_rng(3 * N)
    c = (c0 * (1 + 0.02 * rng.standard_normal((N, N, N)))).astype(np.float32)
    ii = np.arange(N // 2 - 4, N // 2 + 5)
    gy, gx = np.meshgrid(ii, ii, indexing="ij")
    pos = np.stack([gx.ravel() * dx, gy.ravel() * dx, np.full(gx.size, (abl + 3) * dx)], 1)
    amp = np.full((1, pos.shape[0]), 1.0 - 0.5j, dtype=np.complex64)
    k0, eps = R.wavenumber(f, c0, 0.8)
    V = R.potential(c.astype(np.float64), 0.5, 1.1, f, c0, 0.8)
    S = R.deposit((N, N, N), dx, pos, amp[0])
    g = R.green_spectrum((N, N, N), dx, k0, eps)
    win = tuple(R.abl_window(N, abl) for _ in range(3))
    ref = R.solve(V, S, g, 2000, 1e-6, pad=1, windows=win)
    plan = Plan((N, N, N), dx, [f], c0, 0.8)
    plan.set_boundary("periodic")
    plan.set_abl(abl, 9.666)
    plan.set_medium(torch.from_numpy(c).cuda(), alpha0_db=0.5, y=1.1)
    plan.set_source(pos, amp)
    res = plan.solve(2000, 1e-6)
    assert res.status == 0 and ref.status == R.OK
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, "periodic 32^3")


def test_paper_mode_matches_oracle_algorithm_1():
    N, abl = 256, 32
    case = _case(N, abl)
    V, S, g, win = _oracle_inputs(N, abl, *case)
    ref = R.solve_paper_mode(V, S, g, 2000, 1e-5, N // 2, windows=win)
    plan = _plan(N, abl, *case)
    plan.set_criterion("l1_row", N // 2)
    res = plan.solve(2000, 1e-5)
    assert res.status == 0 and ref.status == R.OK
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, "paper mode 256^2")
    compare_history(res.history[0], ref.history, min(int(res.n_terms[0]), ref.n_terms))


def test_paper_homogeneous_case_reproduces_table_3_iteration_count(golden):
    """The paper's own first experiment: 4096^2 periodic grid, dx = 0.02 mm, f = the 55th
    grid harmonic, eps = 0.8 k^2, 501-pixel line source of strength -i 10^6 at column 675 centred on row 2049,
    450-cell sigmoid layer, Eq. 30 on row 2049 below 10^-5.  Table 3 prints 135 iterations for
    the authors' CUDA code and 133 for their CPU code; this path must land within 10 % of them (the two
    printed counts differ by 2; layer geometry and the window on the initial field are readings, DESIGN A4)."""
    from paper_2507_13754_b200.tbs import Plan, grid_harmonic_frequency
    N, dx, c0 = int(golden["n_grid"]), golden["dx_m"], golden["v_f"]
    f = grid_harmonic_frequency(int(golden["f_multiple"]), c0, N, dx)
    assert abs(f - golden["f_hz"]) < 0.5
    plan = Plan((N, N), dx, [f], c0, golden["eps_over_k2"])
    plan.set_boundary("periodic")
    zeta_half_mu = golden["zeta_np_per_cm"] * (golden["abl_cells"] * dx * 100.0) / 2.0
    plan.set_abl(int(golden["abl_cells"]), zeta_half_mu)
    row = int(golden["y_el_row"]) - 1
    plan.set_criterion("l1_row", row)
    plan.set_medium(torch.full((N, N), c0, dtype=torch.float32, device="cuda"), alpha0_db=0.0, y=1.5)
    half = (int(golden["n_el"]) - 1) // 2
    rows = np.arange(row - half, row + half + 1)
    pos = np.stack([np.full(rows.size, golden["x_el_cells"] * dx), rows * dx], 1)
    amp = np.full((1, rows.size), -1j * golden["source_strength"], dtype=np.complex64)
    plan.set_source(pos, amp)
    res = plan.solve(2000, golden["err_threshold"])
    assert res.status == 0
    n = int(res.n_terms[0])
    lo = 0.9 * min(golden["iters_homog_gpu"], golden["iters_homog_cpu"])
    hi = 1.1 * max(golden["iters_homog_gpu"], golden["iters_homog_cpu"])
    assert lo <= n <= hi, n
    # the beam has reached the far absorbing layer: the axial field 60 mm from the source is of the order of
    # the field 10 mm from it (a lossless line source of width 10 mm, Rayleigh distance ~ 17 mm)
    p = res.p[0]
    near = float(p[row, int(golden["x_el_cells"]) + 500].abs())
    far = float(p[row, int(golden["x_el_cells"]) + 3000].abs())
    assert far > 0.2 * near


def _paper_plan(golden, f, c, **medium):
    from paper_2507_13754_b200.tbs import Plan
    N, dx, c0 = int(golden["n_grid"]), golden["dx_m"], golden["v_f"]
    plan = Plan((N, N), dx, [f], c0, golden["eps_over_k2"])
    plan.set_boundary("periodic")
    plan.set_abl(int(golden["abl_cells"]), golden["zeta_np_per_cm"] * (golden["abl_cells"] * dx * 100.0) / 2.0)
    plan.set_criterion("l1_row", int(golden["y_el_row"]) - 1)
    plan.set_medium(c, alpha0_db=0.0, y=1.5, **medium)
    return plan


def _paper_source(golden):
    dx, row = golden["dx_m"], int(golden["y_el_row"]) - 1
    half = (int(golden["n_el"]) - 1) // 2
    rows = np.arange(row - half, row + half + 1)
    pos = np.stack([np.full(rows.size, golden["x_el_cells"] * dx), rows * dx], 1)
    return pos, np.full((1, rows.size), -1j * golden["source_strength"], dtype=np.complex64)


def test_paper_scatterer_cases_follow_table_3(golden):
    """PAPER.md:264 and Table 3: a disc of radius 50 dx on the axis, 40.2 mm from the line
    source, v_s = 1350 / 1650 / 1800 m/s.  The paper's CPU code needs 162 / 155 / 164 iterations (its GPU column
    prints 134 for all three); within 10 % here, and in the same order."""
    from paper_2507_13754_b200.tbs import grid_harmonic_frequency
    N, dx, c0 = int(golden["n_grid"]), golden["dx_m"], golden["v_f"]
    f = grid_harmonic_frequency(int(golden["f_multiple"]), c0, N, dx)
    row = int(golden["y_el_row"]) - 1
    yy, xx = torch.meshgrid(torch.arange(N, device="cuda"), torch.arange(N, device="cuda"), indexing="ij")
    xc = golden["x_el_cells"] + golden["scatterer_dist_m"] / dx
    disc = (xx - xc) ** 2 + (yy - row) ** 2 < golden["scatterer_radius_cells"] ** 2
    pos, amp = _paper_source(golden)
    counts = {}
    for vs in (1350, 1650, 1800):
        c = torch.full((N, N), c0, dtype=torch.float32, device="cuda")
        c[disc] = float(vs)
        plan = _paper_plan(golden, f, c)
        plan.set_source(pos, amp)
        res = plan.solve(2000, golden["err_threshold"])
        assert res.status == 0
        counts[vs] = int(res.n_terms[0])
        ref = golden[f"iters_vs{vs}_cpu"]
        assert 0.9 * ref <= counts[vs] <= 1.1 * ref, (vs, counts[vs], ref)
        del plan
    assert counts[1650] < counts[1350] < counts[1800]


def test_paper_nonlinear_case_follows_table_3_for_five_harmonics(golden):
    """PAPER.md:266 and Table 3: fundamental and harmonics 2-5 of the homogeneous nonlinear
    medium (B/A = 5), eps_h = 0.8 (h k_f)^2, solved one after the other.  The paper prints 135, 228, 306, 368,
    416 iterations (CUDA) and 133, 225, 301, 362, 409 (CPU); each within 10 % here.  The fundamental is rescaled
    to 1 MPa before the harmonic sources are formed (the counts do not depend on the amplitude; complex64 would
    underflow at the paper's source strength by the fourth harmonic)."""
    from paper_2507_13754_b200.tbs import grid_harmonic_frequency, solve_harmonics
    N, dx, c0 = int(golden["n_grid"]), golden["dx_m"], golden["v_f"]
    f1 = grid_harmonic_frequency(int(golden["f_multiple"]), c0, N, dx)
    c = torch.full((N, N), c0, dtype=torch.float32, device="cuda")
    plans = [_paper_plan(golden, h * f1, c, beta=1 + golden["b_over_a"] / 2, rho0=golden["rho_f"]) for h in range(1, 6)]
    plans[0].set_source(*_paper_source(golden))
    st, res = solve_harmonics(plans, 2000, golden["err_threshold"], int(golden["y_el_row"]) - 1, 1.0e6)
    assert st == 0
    counts = [int(r.n_terms[0]) for r in res]
    for h, n in enumerate(counts, start=1):
        lo = 0.9 * min(golden[f"iters_h{h}_gpu"], golden[f"iters_h{h}_cpu"])
        hi = 1.1 * max(golden[f"iters_h{h}_gpu"], golden[f"iters_h{h}_cpu"])
        assert lo <= n <= hi, (h, n)
    # amplitudes fall from harmonic to harmonic
    mags = [float(r.p[0].abs().max()) for r in res]
    assert all(mags[i + 1] < mags[i] for i in range(4))


def test_paper_absorbing_dispersive_case_count_and_attenuation_law(golden):
    """PAPER.md:264 and Table 3: alpha_0 = 5.5e-10 Np (rad/s)^-nu m^-1, nu = 1.5.  The paper applies
    the potential as a k-space multiplier (Eq. 24); this path applies the same medium as a spatial complex
    wavenumber (reading A6, equal on-shell to first order in alpha/k).  The iteration count must land within
    10 % of the printed 132 / 131, and the axial amplitude relative to the lossless run must follow the
    absorption law the multiplier was built from (Eq. 3): exp(-alpha_0 omega^nu d)."""
    from paper_2507_13754_b200.tbs import grid_harmonic_frequency
    N, dx, c0 = int(golden["n_grid"]), golden["dx_m"], golden["v_f"]
    f = grid_harmonic_frequency(int(golden["f_multiple"]), c0, N, dx)
    nu = golden["nu"]
    a0_db = golden["alpha0_si"] * 8.685889638 / 100.0 * (2 * np.pi * 1e6) ** nu      # dB / (MHz^nu cm)
    row, col0 = int(golden["y_el_row"]) - 1, int(golden["x_el_cells"])
    c = torch.full((N, N), c0, dtype=torch.float32, device="cuda")
    fields, counts = [], []
    for a0 in (0.0, a0_db):
        plan = _paper_plan(golden, f, c)
        plan.set_medium(c, alpha0_db=a0, y=nu)
        plan.set_source(*_paper_source(golden))
        res = plan.solve(2000, golden["err_threshold"])
        assert res.status == 0
        counts.append(int(res.n_terms[0]))
        fields.append(res.p[0][row].abs().cpu().numpy())
        del plan
    lo = 0.9 * min(golden["iters_absdisp_gpu"], golden["iters_absdisp_cpu"])
    hi = 1.1 * max(golden["iters_absdisp_gpu"], golden["iters_absdisp_cpu"])
    assert lo <= counts[1] <= hi, counts
    assert counts[1] <= counts[0]                         # Table 3: absorption does not add iterations
    alpha = golden["alpha0_si"] * (2 * np.pi * f) ** nu   # Np/m
    d1, d2 = int(10e-3 / dx), int(50e-3 / dx)
    measured = (fields[1][col0 + d2] / fields[0][col0 + d2]) / (fields[1][col0 + d1] / fields[0][col0 + d1])
    assert abs(measured / np.exp(-alpha * (d2 - d1) * dx) - 1) < 0.02, measured


@pytest.mark.parametrize("boundary", ["pad", "periodic"])
def test_kspace_multiplier_potential_matches_oracle(boundary):
    """Eq. 24 through tbs_set_kspace_absorption, against the oracle's solve_kspace."""
    from paper_2507_13754_b200.tbs import Plan
    N, f, c0 = 128, 1.0e6, 1500.0
    dx = c0 / f / 8.0
    a0, nu, abl = 4.0e-9, 1.5, 16
    rows = np.arange(N // 2 - 12, N // 2 + 13)
    pos = np.stack([np.full(rows.size, (abl + 5) * dx), rows * dx], 1)
    amp = np.full((1, rows.size), -1.0e6j, dtype=np.complex64)
    pad = 1 if boundary == "periodic" else 2
    k0, eps = R.wavenumber(f, c0, 0.8)
    g = R.green_spectrum((pad * N, pad * N), dx, k0, eps)
    VV = R.kspace_potential((pad * N, pad * N), dx, a0, nu, f, c0, 0.8)
    S = R.deposit((N, N), dx, pos, amp[0])
    win = tuple(R.abl_window(N, abl) for _ in range(2))
    ref = R.solve_kspace(S, g, VV, 3000, 1e-6, pad=pad, windows=win)
    plan = Plan((N, N), dx, [f], c0, 0.8)
    plan.set_boundary(boundary)
    plan.set_abl(abl, 9.666)
    plan.set_kspace_absorption(a0, nu)
    plan.set_source(pos, amp)
    res = plan.solve(3000, 1e-6)
    assert res.status == 0 and ref.status == R.OK
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, f"Eq. 24, {boundary}")
    compare_history(res.history[0], ref.history, min(int(res.n_terms[0]), ref.n_terms))


def test_paper_absorbing_rows_of_table_3_with_the_kspace_multiplier(golden):
    """Table 3 in the paper's own formulation (Eq. 24): "absorbing" (lossy operator only)
    133 / 134 iterations, "absorbing-dispersive" 132 / 131; within 10 % here."""
    from paper_2507_13754_b200.tbs import Plan, grid_harmonic_frequency
    N, dx, c0 = int(golden["n_grid"]), golden["dx_m"], golden["v_f"]
    f = grid_harmonic_frequency(int(golden["f_multiple"]), c0, N, dx)
    for dispersive, key in ((False, "abs"), (True, "absdisp")):
        plan = Plan((N, N), dx, [f], c0, golden["eps_over_k2"])
        plan.set_boundary("periodic")
        plan.set_abl(int(golden["abl_cells"]), golden["zeta_np_per_cm"] * (golden["abl_cells"] * dx * 100.0) / 2.0)
        plan.set_criterion("l1_row", int(golden["y_el_row"]) - 1)
        plan.set_kspace_absorption(golden["alpha0_si"], golden["nu"], dispersive)
        plan.set_source(*_paper_source(golden))
        res = plan.solve(2000, golden["err_threshold"])
        assert res.status == 0
        n = int(res.n_terms[0])
        lo = 0.9 * min(golden[f"iters_{key}_gpu"], golden[f"iters_{key}_cpu"])
        hi = 1.1 * max(golden[f"iters_{key}_gpu"], golden[f"iters_{key}_cpu"])
        assert lo <= n <= hi, (key, n)
        del plan


@pytest.mark.parametrize("N,v_s", [(128, 1650.0), (512, 1350.0)])
def test_kspace_multiplier_plus_scatterer_matches_oracle(N, v_s):
    """A disc scatterer (Eqs. 25-26, v_s of Table 3) inside the absorbing-dispersive medium of
    Eq. 24: tbs_set_kspace_absorption + tbs_set_kspace_scatterer on the periodic grid against the
    oracle's solve_kspace(..., Us=...), L2 criterion and the paper's Eq. 30 row criterion."""
    from paper_2507_13754_b200.tbs import Plan, TbsError
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / 8.0
    a0, nu, abl = 4.0e-9, 1.5, N // 8
    rows = np.arange(N // 2 - N // 10, N // 2 + N // 10 + 1)
    pos = np.stack([np.full(rows.size, (abl + 5) * dx), rows * dx], 1)
    amp = np.full((1, rows.size), -1.0e6j, dtype=np.complex64)
    yy, xx = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    disc = (xx - 0.6 * N) ** 2 + (yy - 0.45 * N) ** 2 <= (N / 16) ** 2
    c = np.where(disc, v_s, c0).astype(np.float32)
    k0, eps = R.wavenumber(f, c0, 0.8)
    g = R.green_spectrum((N, N), dx, k0, eps)
    VV = R.kspace_potential((N, N), dx, a0, nu, f, c0, 0.8)
    Us = (2 * np.pi * f / c.astype(np.float64)) ** 2 - k0 * k0
    S = R.deposit((N, N), dx, pos, amp[0])
    win = tuple(R.abl_window(N, abl) for _ in range(2))
    plan = Plan((N, N), dx, [f], c0, 0.8)
    with pytest.raises(TbsError):
        plan.set_kspace_scatterer(torch.from_numpy(c).cuda())      # needs the periodic boundary ...
    plan.set_boundary("periodic")
    with pytest.raises(TbsError):
        plan.set_kspace_scatterer(torch.from_numpy(c).cuda())      # ... and the multiplier
    plan.set_abl(abl, 9.666)
    plan.set_kspace_absorption(a0, nu)
    plan.set_source(pos, amp)
    alone = plan.solve(3000, 1e-6)
    plan.set_kspace_scatterer(torch.from_numpy(c).cuda())
    res = plan.solve(3000, 1e-6)
    ref = R.solve_kspace(S, g, VV, 3000, 1e-6, pad=1, windows=win, Us=Us)
    assert res.status == 0 and ref.status == R.OK
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1, (int(res.n_terms[0]), ref.n_terms)
    compare_fields(res.p[0].cpu().numpy(), ref.p, "Eq. 24 + scatterer")
    compare_history(res.history[0], ref.history, min(int(res.n_terms[0]), ref.n_terms))
    # the scatterer is really in: the field differs from the multiplier-only run by far more than the tolerance
    assert float((res.p - alone.p).abs().max() / alone.p.abs().max()) > 1e-2
    # Eq. 30 on the centre row (the paper's criterion)
    plan.set_criterion("l1_row", N // 2)
    res30 = plan.solve(2000, 1e-5)
    ref30 = R.solve_kspace(S, g, VV, 2000, 1e-5, pad=1, windows=win, row=N // 2, Us=Us)
    assert abs(int(res30.n_terms[0]) - ref30.n_terms) <= 1
    compare_fields(res30.p[0].cpu().numpy(), ref30.p, "Eq. 24 + scatterer, Eq. 30")
    # the multiplier alone again: same result as before the scatterer was set
    plan.set_criterion("l2_grid")
    plan.set_kspace_absorption(a0, nu)
    again = plan.solve(3000, 1e-6)
    assert int(again.n_terms[0]) == int(alone.n_terms[0])
    assert float((again.p - alone.p).abs().max() / alone.p.abs().max()) < 1e-6
