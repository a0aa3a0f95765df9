"""Parity at the sizes BASELINE.json states (north_star: "every config matches the oracle ... same term count at
convergence within +-1"; method PAPER.md:156-160 Eqs. 18-19, stop rule PAPER.md:258-262 / reading A8):

  * 32 Born terms at FULL size for cfg2-cfg5, field and history term by term (the term form makes a
    fixed partial sum exact to compare);
  * converged runs against the live oracle: cfg2 at full size (1024^2), cfg3 at N = 1024 and cfg5 at N = 128 (the
    half-size replicas of SURVEY 8(d)), the 2f chain of cfg4 at N = 1024;
  * cfg3 at full size (2048^2, ~1876 terms) to convergence against the oracle's stored result
    (tests/golden/cfg3_converged.npz, written by tests/golden/make_converged_fields.py, oracle only).
"""
import os

import numpy as np
import pytest

import oracle.tbs_ref as R
import tbs_workloads as W
from parity_util import compare_fields, compare_history, compare_history_converged, gpu_plan, oracle_run

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


# ------------------------------------------------------------------ 32 terms at full size
@pytest.mark.parametrize("maker", [W.cfg2, W.cfg3, W.cfg4, W.cfg5])
def test_full_size_32_terms_match_oracle(maker):
    w = maker()
    terms = 32
    ref = oracle_run(w, terms, 0.0)
    res = gpu_plan(w).solve(terms, 0.0)
    assert int(res.n_terms[0]) == ref.n_terms == terms and res.status == 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, w.name)
    compare_history(res.history[0], ref.history, terms, rtol=1e-4)


# ------------------------------------------------------------------ converged, live oracle
@pytest.mark.parametrize("maker,kw", [(W.cfg2, {}), (W.cfg3, {"N": 1024}), (W.cfg5, {"N": 128})])
def test_converged_field_matches_oracle(maker, kw):
    w = maker(**kw)
    ref = oracle_run(w, w.max_terms, w.tol)
    assert ref.status == 0
    res = gpu_plan(w).solve(w.max_terms, w.tol)
    assert res.status == 0
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1, (int(res.n_terms[0]), ref.n_terms)
    compare_fields(res.p[0].cpu().numpy(), ref.p, w.name)
    n = min(int(res.n_terms[0]), ref.n_terms)
    compare_history_converged(res.history[0], ref.history, n)


def test_second_harmonic_chain_at_1024_matches_oracle():
    """cfg4 (nonlinear, Eq. 28b, 266) at N = 1024: fundamental, 1 MPa rescale, S2, solve at 2 f1."""
    from paper_2507_13754_b200.tbs import Plan, solve_second_harmonic
    w = W.cfg4(N=1024)
    f1 = w.freqs[0]
    ref_row, P0 = 17, w.notes["surface_pressure_pa"]
    plan1 = gpu_plan(w)
    plan2 = Plan(w.shape, w.dx, [2 * f1], w.c0, w.damping)
    plan2.set_medium(torch.from_numpy(w.c).cuda(), alpha0_db=w.alpha0_db, y=w.y, beta=w.beta, rho0=w.rho0)
    st, (r1, r2) = solve_second_harmonic(plan1, plan2, w.max_terms, w.tol, ref_row, P0)
    assert st == 0
    o1 = oracle_run(w, w.max_terms, w.tol)
    p1 = o1.p * (P0 / np.abs(o1.p[ref_row]).max())
    S2 = R.second_harmonic_source(p1, w.beta, w.rho0, w.c0, f1)
    w2 = W.cfg4(N=1024)
    w2.freqs = [2 * f1]
    o2 = oracle_run(w2, w.max_terms, w.tol, S_override=S2)
    assert o1.status == 0 and o2.status == 0
    assert abs(int(r1.n_terms[0]) - o1.n_terms) <= 1 and abs(int(r2.n_terms[0]) - o2.n_terms) <= 1
    compare_fields(r1.p[0].cpu().numpy(), p1, "p1 (1 MPa)")
    compare_fields(r2.p[0].cpu().numpy(), o2.p, "p2")


# ------------------------------------------------------------------ cfg3 at 2048^2 to convergence, stored oracle result
def test_cfg3_full_size_converged_matches_stored_oracle_result():
    path = os.path.join(GOLDEN, "cfg3_converged.npz")
    if not os.path.exists(path):
        pytest.skip("tests/golden/cfg3_converged.npz not generated (tests/golden/make_converged_fields.py cfg3)")
    gold = np.load(path)
    w = W.cfg3()
    assert str(gold["workload"]) == w.name and float(gold["tol"]) == w.tol
    res = gpu_plan(w).solve(w.max_terms, w.tol)
    assert res.status == 0 == int(gold["status"])
    n_ref = int(gold["n_terms"])
    assert abs(int(res.n_terms[0]) - n_ref) <= 1, (int(res.n_terms[0]), n_ref)
    p = res.p[0].cpu().numpy().astype(np.complex128)
    st = int(gold["stride"])
    compare_fields(p[::st, ::st], gold["p_sub"], "cfg3 2048^2 converged (every 16th point)")
    # whole-grid quantities, so the sampled comparison cannot miss a localised error
    assert abs(np.linalg.norm(p) / float(gold["p_norm"]) - 1.0) < 1e-4
    rs = p.sum(axis=1)
    assert np.linalg.norm(rs - gold["p_row_sums"]) <= 1e-4 * np.linalg.norm(gold["p_row_sums"])
    n = min(int(res.n_terms[0]), n_ref)
    compare_history_converged(res.history[0], gold["history"], n)
