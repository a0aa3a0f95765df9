"""CPU-only checks of the boundary and the host logic: the C-ABI library loads and exports every
symbol include/tbs.h declares, argument validation happens before any CUDA work, the frequency
sharding is a partition, and the N>1 timing reduction works over gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    import __graft_entry__ as g
    from paper_2507_13754_b200 import build as b
    b.build()
    from paper_2507_13754_b200 import _lib
    return _lib.load(), _lib


def test_library_exports_every_declared_symbol():
    L, mod = _lib()
    hdr = open(os.path.join(ROOT, "include", "tbs.h")).read()
    declared = set(re.findall(r"\b(tbs_[a-z_0-9]+)\s*\(", hdr))
    declared -= {"tbs_plan", "tbs_status"}
    assert declared, "no declarations parsed"
    for name in sorted(declared):
        assert hasattr(L, name), f"libtbs.so does not export {name}"
    assert declared == set(mod.SYMBOLS), declared ^ set(mod.SYMBOLS)
    assert b"sm_100a" in L.tbs_version()


def test_library_is_built_for_sm_100a_only():
    from paper_2507_13754_b200 import _lib
    out = subprocess.run(["cuobjdump", "-lelf", _lib.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out and "sm_80" not in out


def _create(L, ndim, n, dx=1e-4, freqs=(1e6,), c0=1500.0, damping=0.8):
    h = ctypes.c_void_p()
    nn = (ctypes.c_int32 * 3)(*n)
    ff = (ctypes.c_double * len(freqs))(*freqs)
    st = L.tbs_plan_create(ctypes.byref(h), ndim, nn, dx, len(freqs), ff, c0, damping)
    return st, h


def test_plan_create_validates_before_touching_cuda():
    L, _ = _lib()
    assert _create(L, 1, (64, 64, 1))[0] == -1              # ndim
    assert _create(L, 2, (64, 64, 1), dx=0.0)[0] == -1      # dx
    assert _create(L, 2, (64, 64, 1), damping=0.0)[0] == -1
    assert _create(L, 2, (64, 64, 1), freqs=(0.0,))[0] == -1
    assert _create(L, 2, (48, 64, 1))[0] == -2              # not a power of two
    assert _create(L, 2, (16, 64, 1))[0] == -2              # below 32
    assert _create(L, 2, (8192, 64, 1))[0] == -2            # above 4096 (2-D)
    assert _create(L, 3, (1024, 64, 64))[0] == -2           # above 512 (3-D)
    st, h = _create(L, 2, (64, 64, 1))
    # no CPU fallback: without a device the only acceptable answers are TBS_ERR_CUDA, or TBS_OK on a GPU box
    assert st in (0, -4)
    if st == 0:
        L.tbs_plan_destroy(h)
    else:
        assert not h.value


def test_null_plan_calls_are_rejected():
    L, _ = _lib()
    assert L.tbs_set_abl(None, 4, 9.666) == -1
    assert L.tbs_solve(None, 10, 1e-6, None, None, None, None) == -1
    assert L.tbs_plan_workspace_bytes(None) == 0
    assert L.tbs_last_error(None) == b"null plan"
    L.tbs_plan_destroy(None)


def test_binding_fails_loudly_without_the_library(tmp_path, monkeypatch):
    from paper_2507_13754_b200 import _lib
    monkeypatch.setattr(_lib, "_lib", None)
    monkeypatch.setattr(_lib, "LIB_PATH", str(tmp_path / "missing.so"))
    with pytest.raises(ImportError):
        _lib.load()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2507_13754_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inl", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("the oracle", "").replace("The oracle", ""), (dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2507_13754_b200" not in src and "from paper_2507_13754_b200" not in src


def test_shard_frequencies_is_a_balanced_partition():
    from paper_2507_13754_b200.parallel import shard_frequencies
    for nf in (0, 1, 5, 16, 17):
        for world in (1, 2, 3, 8):
            shards = [shard_frequencies(nf, r, world) for r in range(world)]
            assert sorted(sum(shards, [])) == list(range(nf))
            sizes = [len(s) for s in shards]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_frequencies(4, 2, 2)


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2507_13754_b200.parallel import reduce_timing, shard_frequencies
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
mine = shard_frequencies(5, rank, world)
times, counts = reduce_timing(dist, "cpu", [10.0 + rank, 3.0 - rank], [len(mine), 100 * (rank + 1)])
assert times == [11.0, 3.0], times
assert counts == [5.0, 300.0], counts
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_timing_reduction_over_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29571")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        assert "ok" in out


def test_grid_harmonic_frequency_is_the_papers_number(golden):
    """tbs_grid_harmonic_frequency needs no device: f = 55 v_f/(4096 dx) = 1 007 080 Hz."""
    L, _ = _lib()
    f = L.tbs_grid_harmonic_frequency(int(golden["f_multiple"]), golden["v_f"], 4096, golden["dx_m"])
    assert abs(f - golden["f_hz"]) < 1.0
    assert L.tbs_grid_harmonic_frequency(0, 1500.0, 4096, 2e-5) == 0.0


def test_workspace_calls_reject_null_arguments():
    L, _ = _lib()
    assert L.tbs_plan_set_workspace(None, None, 0) == -1
    assert L.tbs_plan_device_bytes(None) == 0
    assert L.tbs_set_concurrency(None, 2) == -1


_SHARD_WORKER = r"""
import ctypes, os, sys, time
sys.path.insert(0, {root!r})
import numpy as np
import torch, torch.distributed as dist
import tbs_workloads as W
from paper_2507_13754_b200 import _lib
from paper_2507_13754_b200.parallel import reduce_timing, shard_frequencies
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
w = W.cfg5(N=32, nfreq=16)
mine = shard_frequencies(len(w.freqs), rank, world)
freqs = [w.freqs[i] for i in mine]
amp = np.ascontiguousarray(w.src_amp[mine])
assert amp.shape == (len(mine), w.src_pos.shape[0])
# one independent plan per rank over its own block of frequencies: the arguments pass the ABI's validation
# (TBS_OK on a GPU box, TBS_ERR_CUDA here -- never INVALID_ARG / UNSUPPORTED_SIZE); there is no CPU fallback
L = _lib.load()
h = ctypes.c_void_p()
n = (ctypes.c_int32 * 3)(*w.shape[::-1])
ff = (ctypes.c_double * len(freqs))(*freqs)
t0 = time.perf_counter()
st = L.tbs_plan_create(ctypes.byref(h), 3, n, w.dx, len(freqs), ff, w.c0, w.damping)
dt = time.perf_counter() - t0
assert st in (0, -4), st
if st == 0:
    assert L.tbs_plan_workspace_bytes(h) >= 8 * 32 ** 3 * (3 * len(freqs) + 2 * 6)
    L.tbs_plan_destroy(h)
times, counts = reduce_timing(dist, "cpu", [dt, float(rank)], [len(mine), sum(mine)])
assert counts == [16.0, float(sum(range(16)))], counts       # every frequency owned exactly once
assert times[1] == float(world - 1) and times[0] >= dt
dist.barrier()
dist.destroy_process_group()
print("ok", rank, mine)
"""


def test_frequency_shard_path_end_to_end_over_gloo_world_size_2(tmp_path):
    """NEXT-4 host logic: shard the 16-frequency batch, one independent plan per rank, reduce."""
    _lib()
    script = tmp_path / "shard_worker.py"
    script.write_text(_SHARD_WORKER.format(root=ROOT))
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29573")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0, err
        outs.append(out)
    assert "ok 0 [0, 1, 2, 3, 4, 5, 6, 7]" in outs[0] and "ok 1 [8, 9, 10, 11, 12, 13, 14, 15]" in outs[1]


def test_bench_spawns_its_own_ranks_for_gpus_n(monkeypatch):
    """bench.py --gpus N outside torchrun re-launches itself under torch.distributed.run with N ranks."""
    import importlib
    bench = importlib.import_module("bench")
    seen = {}
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "2"])
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert e.value.code == 0
    cmd = seen["cmd"]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=4" in cmd and "--master-addr" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[-4:] == ["--gpus", "4", "--steps", "2"]
