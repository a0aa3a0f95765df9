"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: rel L2 <= 1e-4,
max|dp| <= 1e-3 max|p|, term count within +-1."""
import numpy as np
import pytest

import oracle.tbs_ref as R
import tbs_workloads as W
from parity_util import compare_fields, compare_history, gpu_plan, oracle_run

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _plan(shape, dx=0.25e-3, freqs=(1.0e6,), c0=1500.0, damping=0.8):
    from paper_2507_13754_b200.tbs import Plan
    return Plan(shape, dx, list(freqs), c0, damping)


# ------------------------------------------------------------------ setup kernels (S0a-S0c)
@pytest.mark.parametrize("shape", [(32, 64), (32, 32, 64)])
def test_green_spectrum_matches_oracle(shape):
    plan = _plan(shape)
    g = plan.green_spectrum(0).cpu().numpy()
    k0, eps = R.wavenumber(1.0e6, 1500.0, 0.8)
    ref = R.green_spectrum(tuple(2 * s for s in shape), 0.25e-3, k0, eps)
    assert np.abs(g - ref).max() <= 2e-7 * np.abs(ref).max()


def test_potential_matches_oracle():
    w = W.cfg3(N=64)
    plan = gpu_plan(w)
    V = plan.get_potential(0).cpu().numpy()
    ref = R.potential(w.c.astype(np.float64), w.alpha0_db, w.y, w.freqs[0], w.c0, w.damping)
    assert np.abs(V - ref).max() <= 3e-7 * np.abs(ref).max()
    # alpha0 map path
    amap = torch.full(w.shape, w.alpha0_db, dtype=torch.float32, device="cuda")
    plan.set_medium(torch.from_numpy(w.c).cuda(), alpha0_map=amap, y=w.y)
    assert np.array_equal(plan.get_potential(0).cpu().numpy(), V)


@pytest.mark.parametrize("nd", [2, 3])
def test_source_deposition_matches_oracle(nd):
    rng = np.random.default_rng(nd)
    shape = (32, 64) if nd == 2 else (32, 32, 64)
    dx = 0.25e-3
    n_src = 40
    pos = np.stack([rng.uniform(0, (shape[nd - 1 - a] - 1) * dx, n_src) for a in range(nd)], 1)
    pos[0] = [3 * dx] * nd                       # on a node
    pos[1] = [(shape[nd - 1 - a] - 1) * dx for a in range(nd)]   # last cell
    amp = (rng.standard_normal((2, n_src)) + 1j * rng.standard_normal((2, n_src))).astype(np.complex64)
    plan = _plan(shape, freqs=(1.0e6, 1.3e6))
    plan.set_source(pos, amp)
    for i in range(2):
        S = plan.get_source(i).cpu().numpy()
        ref = R.deposit(shape, dx, pos, amp[i])
        assert np.abs(S - ref).max() <= 1e-6 * np.abs(ref).max()
    with pytest.raises(Exception):
        bad = pos.copy()
        bad[5, 0] = shape[-1] * dx
        plan.set_source(bad, amp)


# ------------------------------------------------------------------ one application of G (S1-S3)
@pytest.mark.parametrize("shape", [(32, 32), (64, 128), (128, 64), (256, 256), (512, 512), (1024, 32),
                                   (32, 1024), (2048, 32), (32, 2048), (4096, 32), (32, 4096),
                                   (32, 32, 32), (32, 64, 128), (128, 32, 64), (512, 32, 32), (32, 512, 32),
                                   (256, 32, 64), (64, 256, 32)])
def test_apply_green_matches_oracle(shape):
    rng = np.random.default_rng(sum(shape))
    x = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
    dx = 1500.0 / 1.0e6 / 6.0
    plan = _plan(shape, dx=dx)
    out = plan.apply_green(0, torch.from_numpy(x).cuda()).cpu().numpy()
    k0, eps = R.wavenumber(1.0e6, 1500.0, 0.8)
    ref = R.apply_G(x.astype(np.complex128), R.green_spectrum(tuple(2 * s for s in shape), dx, k0, eps))
    rel = np.linalg.norm(out - ref) / np.linalg.norm(ref)
    assert rel < 2e-6, rel


def test_apply_green_point_source_is_symmetric_kernel():
    """An impulse gives the discrete Green's function itself: even about the source (property check)."""
    N = 128
    x = torch.zeros((N, N), dtype=torch.complex64, device="cuda")
    x[64, 64] = 1.0
    g = _plan((N, N)).apply_green(0, x).cpu().numpy()
    assert np.abs(g[64, 1:] - g[64, 1:][::-1]).max() < 1e-6 * np.abs(g).max()
    assert np.abs(g[1:, 64] - g[1:, 64][::-1]).max() < 1e-6 * np.abs(g).max()
    assert np.abs(g[1:, 1:] - g[1:, 1:].T).max() < 1e-6 * np.abs(g).max()


# ------------------------------------------------------------------ the series (S0d-S4)
def test_cfg1_full_run_matches_oracle():
    w = W.cfg1()
    ref = oracle_run(w, w.max_terms, w.tol)
    res = gpu_plan(w).solve(w.max_terms, w.tol)
    assert res.status == 0 and ref.status == 0
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, "cfg1")
    n = min(int(res.n_terms[0]), ref.n_terms)
    compare_history(res.history[0], ref.history, n)
    assert np.all(res.history[0][int(res.n_terms[0]) + 1:] == 0)


@pytest.mark.parametrize("graph_batch", [0, 1, 7])
def test_graph_batch_does_not_change_result(graph_batch):
    w = W.cfg1(N=64)
    a = gpu_plan(w, graph_batch=16).solve(500, 1e-6)
    b = gpu_plan(w, graph_batch=graph_batch).solve(500, 1e-6)
    assert int(a.n_terms[0]) == int(b.n_terms[0])
    assert torch.equal(a.p, b.p)


def test_abl_run_matches_oracle():
    w = W.cfg1()
    w.src_pos[:, 1] = 40 * w.dx
    ref = oracle_run(w, 2000, 1e-7, abl_cells=24)
    res = gpu_plan(w, abl_cells=24).solve(2000, 1e-7)
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, "cfg1+abl")


@pytest.mark.parametrize("maker,N", [(W.cfg2, 256), (W.cfg3, 256), (W.cfg3, 512), (W.cfg4, 256)])
def test_scaled_2d_configs_converge_like_oracle(maker, N):
    w = maker(N=N)
    ref = oracle_run(w, w.max_terms, w.tol)
    res = gpu_plan(w).solve(w.max_terms, w.tol)
    assert res.status == ref.status == 0
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, w.name)
    compare_history(res.history[0], ref.history, min(int(res.n_terms[0]), ref.n_terms))


def test_3d_scaled_cfg5_converges_like_oracle():
    w = W.cfg5(N=64)
    ref = oracle_run(w, w.max_terms, w.tol)
    res = gpu_plan(w).solve(w.max_terms, w.tol)
    assert res.status == ref.status == 0
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, w.name)


def test_3d_frequency_batch_matches_per_frequency_oracle():
    w = W.cfg5(N=32, nfreq=16)
    w.freqs = w.freqs[::5]                  # 0.5, 1.0, 1.5, 2.0 MHz (12 .. 3 points per wavelength)
    w.src_amp = w.src_amp[::5]
    res = gpu_plan(w).solve(3000, 1e-6)
    for i in range(len(w.freqs)):
        ref = oracle_run(w, 3000, 1e-6, ifreq=i)
        assert abs(int(res.n_terms[i]) - ref.n_terms) <= 1, (i, res.n_terms, ref.n_terms)
        compare_fields(res.p[i].cpu().numpy(), ref.p, f"batch f{i}")


def test_rectangular_grids():
    w = W.cfg3(N=128)
    w.shape = (64, 128)
    w.c = np.ascontiguousarray(w.c[:64])
    w.src_pos[:, 1] = 10 * w.dx
    ref = oracle_run(w, 3000, 1e-6)
    res = gpu_plan(w).solve(3000, 1e-6)
    assert abs(int(res.n_terms[0]) - ref.n_terms) <= 1
    compare_fields(res.p[0].cpu().numpy(), ref.p, "64x128")
