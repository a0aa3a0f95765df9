"""GPU parity of the convergent Born series scheme (tbs_set_scheme) against the oracle."""
import numpy as np
import pytest
import torch

import oracle.tbs_ref as R
from parity_util import compare_fields, compare_history

pytestmark = pytest.mark.gpu


def _strong_disc(N, ratio=1.3):
    """Lossless water with a slow disc of radius N/4: k^2/k0^2 - 1 = ratio^2 - 1 = 0.69 < damping 0.8, far beyond
    what the traditional series tolerates (rho(G V) > 1), inside the CBS condition of PAPER.md:445."""
    f, c0 = 1.0e6, 1500.0
    dx = c0 / f / 6.0
    ax = np.arange(N) - (N - 1) / 2
    yy, xx = np.meshgrid(ax, ax, indexing="ij")
    c = np.full((N, N), c0, dtype=np.float32)
    c[np.hypot(xx, yy - N / 8) < N / 4] = c0 / ratio
    cols = np.arange(N // 4, 3 * N // 4)
    pos = np.stack([cols * dx, np.full(cols.size, 4 * dx)], 1)
    amp = np.ones((1, cols.size), dtype=np.complex64)
    return f, c0, dx, c, pos, amp


def _plan(N, scheme):
    from paper_2507_13754_b200.tbs import Plan
    f, c0, dx, c, pos, amp = _strong_disc(N)
    plan = Plan((N, N), dx, [f], c0, 0.8)
    plan.set_scheme(scheme)
    plan.set_medium(torch.from_numpy(c).cuda(), alpha0_db=0.0, y=1.5)
    plan.set_source(pos, amp)
    return plan


def test_cbs_matches_oracle_where_born_does_not_converge():
    N = 64
    f, c0, dx, c, pos, amp = _strong_disc(N)
    k0, eps = R.wavenumber(f, c0, 0.8)
    V = R.potential(c.astype(np.float64), 0.0, 1.5, f, c0, 0.8)
    g = R.green_spectrum((2 * N, 2 * N), dx, k0, eps)
    S = R.deposit((N, N), dx, pos, amp[0])
    ref = R.solve_cbs(V, S, g, eps, 4000, 1e-6)
    assert ref.status == R.OK
    res = _plan(N, "cbs").solve(4000, 1e-6)
    assert res.status == 0
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, "CBS 64^2")
    compare_history(res.history[0], ref.history, min(int(res.n_terms[0]), ref.n_terms))
    # the traditional series on the same medium is not converging
    born = _plan(N, "born").solve(300, 1e-6)
    assert born.status != 0


def test_cbs_equals_born_for_homogeneous_lossless_medium():
    """V = -i eps => gamma = 1: both schemes produce the same terms (checked on the GPU path itself)."""
    from paper_2507_13754_b200.tbs import Plan
    N, f, c0 = 128, 1.0e6, 1500.0
    dx = c0 / f / 6.0
    c = np.full((N, N), c0, dtype=np.float32)
    pos = np.array([[40.3 * dx, 8 * dx], [70 * dx, 8 * dx]])
    amp = np.array([[1.0, 0.5j]], dtype=np.complex64)
    out = []
    for scheme in ("born", "cbs"):
        plan = Plan((N, N), dx, [f], c0, 0.8)
        plan.set_scheme(scheme)
        plan.set_medium(torch.from_numpy(c).cuda(), alpha0_db=0.0, y=1.5)
        plan.set_source(pos, amp)
        out.append(plan.solve(2000, 1e-6))
    assert int(out[0].n_terms[0]) == int(out[1].n_terms[0])
    a, b = out[0].p[0].cpu().numpy(), out[1].p[0].cpu().numpy()
    assert np.linalg.norm(a - b) <= 2e-6 * np.linalg.norm(a)


def test_cbs_large_grid_satisfies_the_lippmann_schwinger_equation():
    """256^2 (no oracle run at this size: ~10^4 terms): the converged field must satisfy p = G(V p) + G S
    (Eq. 17), checked with the plan's own single application of G.  The residual is the next
    term divided by gamma, so it sits at the stopping tolerance."""
    N = 256
    f, c0, dx, c, pos, amp = _strong_disc(N)
    plan = _plan(N, "cbs")
    res = plan.solve(40000, 1e-6)
    assert res.status == 0, (res.status, res.n_terms)
    p = res.p[0]
    V = plan.get_potential(0)
    S = plan.get_source(0)
    rhs = plan.apply_green(0, V * p + S)
    rel = float(torch.linalg.norm(p - rhs) / torch.linalg.norm(p))
    assert rel < 2e-5, rel
