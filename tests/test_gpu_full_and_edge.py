"""GPU parity at BASELINE.json's full sizes (partial sums after a few terms, which the term form makes
exact to compare), the nonlinear 2f solve, host-buffer entry points, and the degenerate cases."""
import numpy as np
import pytest

import oracle.tbs_ref as R
import tbs_workloads as W
from parity_util import compare_fields, compare_history, gpu_plan, oracle_run

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


# ------------------------------------------------------------------ full sizes, fixed number of terms
@pytest.mark.parametrize("maker,terms", [(W.cfg2, 6), (W.cfg3, 4), (W.cfg4, 2)])
def test_full_size_2d_partial_sums_match_oracle(maker, terms):
    """Same launch configuration bench.py times (full N), p and history after `terms` terms."""
    w = maker()
    ref = oracle_run(w, terms, 0.0)
    res = gpu_plan(w).solve(terms, 0.0)
    assert int(res.n_terms[0]) == ref.n_terms == terms and res.status == 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, w.name)
    compare_history(res.history[0], ref.history, terms, rtol=1e-4)


def test_full_size_3d_256_partial_sum_matches_oracle():
    w = W.cfg5()
    terms = 2
    ref = oracle_run(w, terms, 0.0)
    res = gpu_plan(w).solve(terms, 0.0)
    assert int(res.n_terms[0]) == terms
    compare_fields(res.p[0].cpu().numpy(), ref.p, w.name)
    compare_history(res.history[0], ref.history, terms, rtol=1e-4)


def test_cfg3_full_size_converged_field_properties():
    """At full size the oracle cannot run ~1900 terms in a test; check properties that hold at any
    size: the converged p satisfies the fixed-point equation p = G(V p + S) to the stop tolerance,
    evaluated with the oracle's G on sampled rows via one full apply (a few seconds)."""
    w = W.cfg3(N=1024)
    plan = gpu_plan(w)
    res = plan.solve(w.max_terms, w.tol)
    assert res.status == 0
    p = res.p[0].cpu().numpy().astype(np.complex128)
    f = w.freqs[0]
    k0, eps = R.wavenumber(f, w.c0, w.damping)
    g = R.green_spectrum(tuple(2 * s for s in w.shape), w.dx, k0, eps)
    V = R.potential(w.c.astype(np.float64), w.alpha0_db, w.y, f, w.c0, w.damping)
    S = R.deposit(w.shape, w.dx, w.src_pos, w.src_amp[0])
    resid = R.apply_G(V * p + S, g) - p
    # ||G V u_n|| <= ||u_n|| / (1 - rho) ~ tol ||p|| x tail sum; allow 100x tol
    assert np.linalg.norm(resid) / np.linalg.norm(p) < 100 * w.tol
    h = res.history[0][: int(res.n_terms[0]) + 1]
    assert np.all(h[1:] > 0) and h[-1] < w.tol <= h[-2]
    tail = h[-50:]
    assert np.all(tail[1:] / tail[:-1] < 1.0)          # geometric convergence at the end


# ------------------------------------------------------------------ nonlinear 2f (S6)
def test_second_harmonic_matches_oracle():
    from paper_2507_13754_b200.tbs import Plan, solve_second_harmonic
    w = W.cfg4(N=256)
    f1 = w.freqs[0]
    ref_row, P0 = 17, 1.0e6
    plan1 = gpu_plan(w)
    plan2 = Plan(w.shape, w.dx, [2 * f1], w.c0, w.damping)
    plan2.set_medium(torch.from_numpy(w.c).cuda(), alpha0_db=w.alpha0_db, y=w.y, beta=w.beta, rho0=w.rho0)
    st, (r1, r2) = solve_second_harmonic(plan1, plan2, 4000, 1e-6, ref_row, P0)
    assert st == 0
    # oracle: solve f1, rescale to 1 MPa on the reference row, S2 (Eq. 28b), solve 2 f1
    o1 = oracle_run(w, 4000, 1e-6)
    p1 = o1.p * (P0 / np.abs(o1.p[ref_row]).max())
    S2 = R.second_harmonic_source(p1, w.beta, w.rho0, w.c0, f1)
    w2 = W.cfg4(N=256)
    w2.freqs = [2 * f1]
    o2 = oracle_run(w2, 4000, 1e-6, S_override=S2)
    assert abs(int(r1.n_terms[0]) - o1.n_terms) <= 1 and abs(int(r2.n_terms[0]) - o2.n_terms) <= 1
    compare_fields(r1.p[0].cpu().numpy(), p1, "p1 (1 MPa)")
    compare_fields(r2.p[0].cpu().numpy(), o2.p, "p2")
    assert abs(np.abs(r1.p[0, ref_row].cpu().numpy()).max() - P0) < 1e-3 * P0


def test_harmonics_up_to_fifth_match_oracle():
    """NEXT row 1: harmonics 3-5, Eqs. 28c-28e, solved one after the other
    with eps_h = damping (h k_f)^2 from the fields of the lower harmonics."""
    from paper_2507_13754_b200.tbs import Plan, solve_harmonics
    w = W.cfg4(N=128)
    f1 = w.freqs[0]
    ref_row, P0, NH = 17, 1.0e6, 5
    plans = [gpu_plan(w)]
    for h in range(2, NH + 1):
        pl = Plan(w.shape, w.dx, [h * f1], w.c0, w.damping)
        pl.set_medium(torch.from_numpy(w.c).cuda(), alpha0_db=w.alpha0_db, y=w.y, beta=w.beta, rho0=w.rho0)
        plans.append(pl)
    st, res = solve_harmonics(plans, 4000, 1e-6, ref_row, P0)
    assert st == 0
    o1 = oracle_run(w, 4000, 1e-6)
    fields = [o1.p * (P0 / np.abs(o1.p[ref_row]).max())]
    terms = [o1.n_terms]
    for h in range(2, NH + 1):
        S = R.harmonic_source(h, fields, w.beta, w.rho0, w.c0, f1)
        wh = W.cfg4(N=128)
        wh.freqs = [h * f1]
        oh = oracle_run(wh, 4000, 1e-6, S_override=S)
        fields.append(oh.p)
        terms.append(oh.n_terms)
    for h in range(NH):
        assert abs(int(res[h].n_terms[0]) - terms[h]) <= 1, (h + 1, res[h].n_terms, terms[h])
        compare_fields(res[h].p[0].cpu().numpy(), fields[h], f"harmonic {h + 1}")
    # higher harmonics need more terms (eps_h grows as h^2, Table 4 shows the same trend)
    assert terms[4] > terms[1] > terms[0]


# ------------------------------------------------------------------ host-buffer entry points
def test_host_entry_points_equal_device_entry_points():
    w = W.cfg3(N=128)
    plan = gpu_plan(w)
    a = plan.solve(300, 1e-6)
    from paper_2507_13754_b200.tbs import Plan
    plan_h = Plan(w.shape, w.dx, w.freqs, w.c0, w.damping)
    plan_h.set_medium_host(w.c, alpha0_db=w.alpha0_db, y=w.y)
    plan_h.set_source(w.src_pos, w.src_amp)
    b = plan_h.solve_host(300, 1e-6)
    assert int(a.n_terms[0]) == int(b.n_terms[0])
    # source deposition uses float atomics (order not fixed), so two plans agree to rounding only
    pa = a.p.cpu().numpy()
    assert np.abs(pa - b.p).max() <= 1e-5 * np.abs(pa).max()
    assert np.allclose(a.history, b.history, rtol=1e-5)
    assert b.launches > 0 and b.loop_ms > 0


# ------------------------------------------------------------------ degenerate and error cases
def test_zero_potential_stops_after_one_zero_term():
    w = W.cfg1(N=64)
    plan = gpu_plan(w)
    plan.set_potential(0, torch.zeros(w.shape, dtype=torch.complex64, device="cuda"))
    res = plan.solve(50, 1e-6)
    assert res.status == 0 and int(res.n_terms[0]) == 1 and res.history[0][1] == 0.0
    u0 = plan.apply_green(0, plan.get_source(0))
    assert torch.equal(res.p[0], u0)


def test_raw_potential_roundtrip_and_equivalence():
    w = W.cfg3(N=64)
    plan = gpu_plan(w)
    a = plan.solve(200, 1e-6)
    V = plan.get_potential(0)
    plan.set_potential(0, V)
    b = plan.solve(200, 1e-6)
    assert int(a.n_terms[0]) == int(b.n_terms[0])
    rel = (a.p - b.p).abs().max() / a.p.abs().max()
    assert float(rel) < 1e-5


def test_max_terms_zero_returns_u0_not_converged():
    w = W.cfg1(N=64)
    plan = gpu_plan(w)
    res = plan.solve(0, 1e-6)
    assert res.status == 1 and int(res.n_terms[0]) == 0 and res.history[0][0] == 1.0
    ref = oracle_run(w, 0, 1e-6)
    compare_fields(res.p[0].cpu().numpy(), ref.p, "u0")


def test_not_converged_at_cap_keeps_valid_field():
    w = W.cfg1(N=64)
    ref = oracle_run(w, 25, 1e-9)
    res = gpu_plan(w).solve(25, 1e-9)
    assert res.status == 1 == ref.status and int(res.n_terms[0]) == 25
    compare_fields(res.p[0].cpu().numpy(), ref.p, "capped")


def test_not_ready_and_bad_arguments():
    from paper_2507_13754_b200.tbs import Plan, TbsError
    plan = Plan((64, 64), 1e-4, [1e6], 1500.0, 0.8)
    with pytest.raises(TbsError) as e:
        plan.solve(10, 1e-6)
    assert e.value.status == -3
    with pytest.raises(TbsError):
        Plan((48, 64), 1e-4, [1e6], 1500.0, 0.8)
    with pytest.raises(TbsError):
        plan.set_abl(40)                      # wider than half the grid
    c = torch.full((64, 64), 1500.0, device="cuda")
    with pytest.raises(TbsError):
        plan.set_medium(c, alpha0_db=0.5, y=1.0)    # y = 1 excluded
    assert plan.workspace_bytes() >= 64 * 64 * 8 * 5
