"""Writes tests/golden/<name>_converged.npz: the ORACLE's converged Born series of a full-size workload.

Calls only oracle/ and the seeded input generator (tbs_workloads.py); no value here ever comes from the CUDA path.
The full-size runs take minutes of CPU (cfg3, 2-D 2048^2: 1876 terms of a padded 4096^2 complex128 transform
pair), which is why their result is stored instead of being recomputed inside the GPU test:

    python tests/golden/make_converged_fields.py cfg3            # ~10-25 min on 8-16 cores

Stored: n_terms, status, the full history, the field on a regular sub-grid (every `stride`-th point of every
axis, complex128) and, so the sampled comparison still sees the whole grid, the L2 norm of the full field and its
row sums.  Method: SURVEY 8(c) definition (Eqs. 18-19, stop rule PAPER.md:258-262 / reading A8).
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle.tbs_ref as R          # noqa: E402
import tbs_workloads as W           # noqa: E402

STRIDE = {"cfg3": 16}


def main(name):
    w = {"cfg3": W.cfg3}[name]()
    f = w.freqs[0]
    k0, eps = R.wavenumber(f, w.c0, w.damping)
    g = R.green_spectrum(tuple(2 * s for s in w.shape), w.dx, k0, eps)
    V = R.potential(w.c.astype(np.float64), w.alpha0_db, w.y, f, w.c0, w.damping)
    S = R.deposit(w.shape, w.dx, w.src_pos, w.src_amp[0])
    t0 = time.time()
    res = R.solve(V, S, g, w.max_terms, w.tol)
    dt = time.time() - t0
    st = STRIDE[name]
    sl = tuple(slice(None, None, st) for _ in w.shape)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"{name}_converged.npz")
    np.savez_compressed(out, workload=w.name, n_terms=res.n_terms, status=res.status, history=res.history,
                        stride=st, p_sub=res.p[sl], p_norm=np.linalg.norm(res.p),
                        p_row_sums=res.p.reshape(res.p.shape[0], -1).sum(axis=1), tol=w.tol,
                        oracle_seconds=dt, oracle_threads=R.num_threads())
    print(f"{w.name}: {res.n_terms} terms, status {res.status}, {dt:.0f} s on {R.num_threads()} threads -> {out}")


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "cfg3")
