"""The boundary beyond the plain solve: caller-owned workspace, re-use of one plan with
growing max_terms, the divergence guard, the state rules of the k-space potential, and the frequency batch solved
two members at a time against the per-frequency oracle."""
import numpy as np
import pytest

import oracle.tbs_ref as R
import tbs_workloads as W
from parity_util import compare_fields, compare_history, gpu_plan, oracle_run

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _bare_plan(w):
    from paper_2507_13754_b200.tbs import Plan
    return Plan(w.shape, w.dx, w.freqs, w.c0, w.damping)


def _setup(plan, w):
    plan.set_medium(torch.from_numpy(w.c).cuda(), alpha0_db=w.alpha0_db, y=w.y, beta=w.beta, rho0=w.rho0)
    plan.set_source(w.src_pos, w.src_amp)


# ------------------------------------------------------------------ workspace (tbs_plan_set_workspace)
@pytest.mark.parametrize("maker,kw", [(W.cfg3, {"N": 128}), (W.cfg5, {"N": 32})])
def test_solve_in_a_torch_owned_workspace(maker, kw):
    w = maker(**kw)
    plan = _bare_plan(w)
    need = plan.workspace_bytes()
    n = w.n_points
    # V, S, p per frequency + W1 (+ W2 in 3-D), known before anything is allocated
    assert need >= 8 * n * (3 + 2 + (4 if w.ndim == 3 else 0))
    assert plan.device_bytes() < need           # nothing of the workspace is allocated yet: tables only
    before = torch.cuda.memory_allocated()
    buf = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    off = (-buf.data_ptr()) % 256
    plan.set_workspace(buf[off:off + need])
    _setup(plan, w)
    res = plan.solve(300, 1e-6)
    assert plan.device_bytes() < need           # the plan never allocated a workspace of its own
    ref = gpu_plan(w).solve(300, 1e-6)          # a plan that owns its workspace
    assert int(res.n_terms[0]) == int(ref.n_terms[0]) and res.status == ref.status
    rel = (res.p - ref.p).abs().max() / ref.p.abs().max()
    assert float(rel) < 1e-5                    # deposition atomics: the two plans agree to rounding
    o = oracle_run(w, 300, 1e-6)
    compare_fields(res.p[0].cpu().numpy(), o.p, "workspace")
    # the running field lives in the caller's buffer: V, S, p of frequency 0 come first
    p_in_ws = buf[off:off + need][16 * n: 24 * n].view(torch.complex64).reshape(w.shape)
    assert torch.equal(p_in_ws, res.p[0])
    del plan
    assert torch.cuda.memory_allocated() >= before


def test_set_workspace_rejects_bad_buffers():
    from paper_2507_13754_b200.tbs import TbsError
    w = W.cfg1(N=64)
    plan = _bare_plan(w)
    need = plan.workspace_bytes()
    with pytest.raises(TbsError):
        plan.set_workspace(torch.empty(need // 2, dtype=torch.uint8, device="cuda"))
    buf = torch.empty(need + 512, dtype=torch.uint8, device="cuda")
    off = (-buf.data_ptr()) % 256
    with pytest.raises(TbsError):
        plan.set_workspace(buf[off + 8: off + 8 + need])       # misaligned
    # rebinding drops medium and source
    plan.set_workspace(buf[off:off + need])
    _setup(plan, w)
    plan.solve(5, 1e-6)
    buf2 = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    off2 = (-buf2.data_ptr()) % 256
    plan.set_workspace(buf2[off2:off2 + need])
    with pytest.raises(TbsError) as e:
        plan.solve(5, 1e-6)
    assert e.value.status == -3


# ------------------------------------------------------------------ one plan, growing max_terms (graph re-use)
def test_same_plan_with_growing_max_terms_and_profile_in_between():
    w = W.cfg3(N=128)
    plan = gpu_plan(w)
    a = plan.solve(40, 1e-6)                    # capped: TBS_NOT_CONVERGED
    assert a.status == 1 and int(a.n_terms[0]) == 40
    b = plan.solve(2000, 1e-6)                  # the natural follow-up; history buffers grow
    fresh = gpu_plan(w).solve(2000, 1e-6)
    assert b.status == 0 == fresh.status and int(b.n_terms[0]) == int(fresh.n_terms[0])
    assert torch.equal(b.p, fresh.p) or float((b.p - fresh.p).abs().max() / fresh.p.abs().max()) < 1e-5
    assert np.allclose(b.history, fresh.history, rtol=1e-5)
    assert np.allclose(a.history[0][:41], b.history[0][:41], rtol=1e-5)
    ms = plan.profile_term(0, reps=200)         # reps + warm-up beyond the current history capacity? no: 200 < 2000
    assert ms[0] > 0 and ms[1] > 0
    c = plan.solve(2000, 1e-6)
    assert c.status == 0 and int(c.n_terms[0]) == int(fresh.n_terms[0])
    assert np.allclose(c.history, fresh.history, rtol=1e-5)
    plan2 = gpu_plan(w)
    plan2.solve(10, 1e-6)
    plan2.profile_term(0, reps=64)              # grows the buffers under a captured graph
    d = plan2.solve(2000, 1e-6)
    assert d.status == 0 and np.allclose(d.history, fresh.history, rtol=1e-5)


# ------------------------------------------------------------------ divergence guard
def test_strongly_divergent_potential_is_reported():
    w = W.cfg1(N=64)
    plan = gpu_plan(w)
    k0, eps = R.wavenumber(w.freqs[0], w.c0, w.damping)
    plan.set_potential(0, torch.full(w.shape, 30.0 * k0 * k0, dtype=torch.complex64, device="cuda"))
    res = plan.solve(3000, 1e-12)
    assert res.status == -5
    assert "diverged" in plan._L.tbs_last_error(plan._h).decode()
    assert int(res.n_terms[0]) < 200


def test_slowly_divergent_potential_is_reported_long_before_the_cap():
    """A uniform real offset of +35 % of k0^2 over a 128^2 box makes ||GV|| > 1: ||u_n|| grows by a few
    per cent per term and never overflows within the cap; the guard stops it once it has grown a million-fold."""
    w = W.cfg1(N=128)
    k0, eps = R.wavenumber(w.freqs[0], w.c0, w.damping)
    V = np.full(w.shape, 0.35 * k0 * k0 - 1j * eps, dtype=np.complex64)
    o = R.solve(V.astype(np.complex128), R.deposit(w.shape, w.dx, w.src_pos, w.src_amp[0]),
                R.green_spectrum(tuple(2 * s for s in w.shape), w.dx, k0, eps), 400, 1e-9)
    u0 = R.apply_G(R.deposit(w.shape, w.dx, w.src_pos, w.src_amp[0]).astype(np.complex128),
                   R.green_spectrum(tuple(2 * s for s in w.shape), w.dx, k0, eps))
    # the oracle only caps: after 400 terms the term norm has grown 10^9-fold and is still growing
    assert o.status == 1 and np.linalg.norm(o.u_last) > 1e8 * np.linalg.norm(u0)
    plan = gpu_plan(w)
    plan.set_potential(0, torch.from_numpy(V).cuda())
    res = plan.solve(20000, 1e-9)
    assert res.status == -5 and 100 < int(res.n_terms[0]) < 400      # 10^6-fold at ~5.8 % per term
    h = res.history[0][: int(res.n_terms[0]) + 1]
    assert np.all(np.isfinite(h))
    # up to the stop the two sides agree term by term (the guard changes when it stops, not what it computes)
    n = min(int(res.n_terms[0]), o.n_terms)
    compare_history(res.history[0], o.history, n, rtol=1e-3)


# ------------------------------------------------------------------ k-space potential state (Eq. 24 is not combined)
def test_kspace_potential_state_rules():
    from paper_2507_13754_b200.tbs import TbsError
    w = W.cfg2(N=128)
    plan = gpu_plan(w)
    base = plan.solve(400, 1e-6)
    plan.set_kspace_absorption(5.5e-10, 1.5)
    with pytest.raises(TbsError):
        plan.set_scheme("cbs")                   # not combined with Eq. 24
    k = plan.solve(400, 1e-6)
    assert k.status == 0
    # a spatial potential replaces the multiplier: back to the first result
    plan.set_medium(torch.from_numpy(w.c).cuda(), alpha0_db=w.alpha0_db, y=w.y)
    again = plan.solve(400, 1e-6)
    assert int(again.n_terms[0]) == int(base.n_terms[0])
    assert float((again.p - base.p).abs().max() / base.p.abs().max()) < 1e-6
    plan.set_scheme("cbs")
    with pytest.raises(TbsError):
        plan.set_kspace_absorption(5.5e-10, 1.5)


# ------------------------------------------------------------------ frequency batch, two members at a time (S5)
@pytest.mark.parametrize("maker,kw,nf", [(W.cfg5, {"N": 64}, 16), (W.cfg3, {"N": 256}, 5)])
def test_frequency_batch_solved_together_matches_per_frequency_oracle(maker, kw, nf):
    if maker is W.cfg5:
        w = maker(nfreq=nf, **kw)
    else:
        w = maker(**kw)
        w.freqs = [w.freqs[0] * s for s in (0.5, 0.7, 1.0, 0.6, 0.8)]
        w.src_amp = np.repeat(w.src_amp, nf, axis=0)
    plan = gpu_plan(w)
    res = plan.solve(w.max_terms, w.tol)          # default: two members in flight
    assert res.status == 0
    plan.set_concurrency(4)
    four = plan.solve(w.max_terms, w.tol)         # four in flight: slots three and four are the plan's own
    assert np.array_equal(res.n_terms, four.n_terms)
    assert float((res.p - four.p).abs().max() / four.p.abs().max()) < 1e-6
    plan.set_concurrency(1)
    seq = plan.solve(w.max_terms, w.tol)          # one after the other
    assert np.array_equal(res.n_terms, seq.n_terms)
    assert float((res.p - seq.p).abs().max() / seq.p.abs().max()) < 1e-6
    assert np.allclose(res.history, seq.history, rtol=1e-6)
    for i in range(nf):
        ref = oracle_run(w, w.max_terms, w.tol, ifreq=i)
        assert abs(int(res.n_terms[i]) - ref.n_terms) <= 1, (i, int(res.n_terms[i]), ref.n_terms)
        compare_fields(res.p[i].cpu().numpy(), ref.p, f"{w.name} member {i}")
        n = min(int(res.n_terms[i]), ref.n_terms)
        compare_history(res.history[i], ref.history, n, rtol=2e-3)


# ------------------------------------------------------------------ launch switches do not change results
def test_launch_overlap_and_plain_launches_give_the_same_series():
    """tbs_set_launch_overlap (programmatic dependent launch: every kernel orders its memory accesses behind its
    predecessor with griddepcontrol.wait) and tbs_set_graph_batch(0) (no CUDA graph) change how the kernels of a
    term are launched, not what they compute."""
    for w in (W.cfg3(N=256), W.cfg5(N=32)):
        base = gpu_plan(w).solve(w.max_terms, w.tol)
        assert base.status == 0
        for setup in ("overlap", "nograph", "overlap+nograph"):
            plan = gpu_plan(w)
            if "overlap" in setup:
                plan.set_launch_overlap(True)
            if "nograph" in setup:
                plan.set_graph_batch(0)
            res = plan.solve(w.max_terms, w.tol)
            assert res.status == 0 and int(res.n_terms[0]) == int(base.n_terms[0]), setup
            assert float((res.p - base.p).abs().max() / base.p.abs().max()) < 1e-5, setup
            assert np.allclose(res.history, base.history, rtol=1e-5), setup


# ------------------------------------------------------------------ resume after the cap
@pytest.mark.parametrize("maker,kw", [(W.cfg3, {"N": 256}), (W.cfg5, {"N": 32})])
def test_resume_after_the_cap_equals_one_uninterrupted_solve(maker, kw):
    from paper_2507_13754_b200.tbs import TbsError
    w = maker(**kw)
    full = gpu_plan(w).solve(w.max_terms, w.tol)
    assert full.status == 0
    n = int(full.n_terms[0])
    plan = gpu_plan(w)
    a = plan.solve(37, w.tol)                       # stops at its cap in the middle of a graph batch
    assert a.status == 1 and int(a.n_terms[0]) == 37
    b = plan.solve_resume(n // 2, w.tol)            # still capped; the history buffers grow
    assert b.status == 1 and int(b.n_terms[0]) == n // 2
    assert np.array_equal(b.history[0][:38], a.history[0][:38])
    c = plan.solve_resume(w.max_terms, w.tol)       # to convergence
    assert c.status == 0 and int(c.n_terms[0]) == n
    # same kernels, same order of operations; the two plans' sources differ by the rounding of the deposition's
    # float atomics where sub-sources share cells (3-D), and the norms by the order of the fp64 atomics across CTAs
    assert float((c.p - full.p).abs().max() / full.p.abs().max()) < 1e-5
    assert np.allclose(c.history, full.history, rtol=1e-5, atol=0)
    with pytest.raises(TbsError) as e:
        plan.solve_resume(w.max_terms, w.tol)       # nothing capped to continue
    assert e.value.status == -3
    d = plan.solve(20, w.tol)
    assert d.status == 1
    plan.set_abl(4)                                 # any change in between invalidates the state
    with pytest.raises(TbsError):
        plan.solve_resume(100, w.tol)
    ref = oracle_run(w, w.max_terms, w.tol)
    assert abs(n - ref.n_terms) <= 1
    compare_fields(c.p[0].cpu().numpy(), ref.p, "resumed")
