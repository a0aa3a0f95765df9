"""Compile the CUDA library in-tree for sm_100a: ``python -m paper_2507_13754_b200.build``.

``csrc/tbs.cu`` (C ABI, plan, setup kernels, term loop) and ``csrc/inst.cu`` once per transform length
(``-DTBS_N=32 ... 4096``: the Born-term kernels of that length) are compiled side by side and linked into
``libtbs.so``.  Objects are cached under ``build/`` (git-ignored) and rebuilt when any source is newer.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
OUT = os.path.join(HERE, "libtbs.so")
SIZES = (32, 64, 128, 256, 512, 1024, 2048, 4096)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def deps():
    out = []
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        out += [os.path.join(root, f) for f in os.listdir(root)]
    return out


def units():
    """(object path, source, extra flags) of every translation unit."""
    u = [(os.path.join(OBJ, "tbs.o"), os.path.join(CSRC, "tbs.cu"), [])]
    u += [(os.path.join(OBJ, f"inst_{n}.o"), os.path.join(CSRC, "inst.cu"), [f"-DTBS_N={n}"]) for n in SIZES]
    return u


def build(force: bool = False, verbose: bool = False, sizes=None) -> str:
    """sizes: rebuild only these transform lengths' objects (development aid); None = all that are stale."""
    newest = max(os.path.getmtime(p) for p in deps())
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= newest:
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    todo = []
    for obj, src, extra in units():
        stale = force or not os.path.exists(obj) or os.path.getmtime(obj) < newest
        if sizes is not None and extra and int(extra[0].split("=")[1]) not in sizes and os.path.exists(obj):
            stale = False
        if stale:
            todo.append([nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + extra + ["-c", src, "-o", obj])
    with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as ex:
        for r in ex.map(lambda c: subprocess.run(c, capture_output=True, text=True), todo):
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                raise subprocess.CalledProcessError(r.returncode, r.args)
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", OUT] + [u[0] for u in units()],
                   check=True)
    return OUT


if __name__ == "__main__":
    only = [int(a.split("=")[1]) for a in sys.argv if a.startswith("--sizes=")]
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, sizes=only or None))
