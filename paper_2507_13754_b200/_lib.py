"""Loader for the in-tree CUDA library ``libtbs.so`` (C ABI declared in include/tbs.h).

There is no CPU fallback and no other implementation: if the shared library is missing or does
not load, importing the binding fails loudly.  Build it with ``python -m paper_2507_13754_b200.build``
(or ``__graft_entry__.build()``).
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtbs.so")

# every symbol include/tbs.h declares
SYMBOLS = [
    "tbs_version", "tbs_plan_create", "tbs_plan_destroy", "tbs_plan_workspace_bytes", "tbs_plan_set_workspace",
    "tbs_plan_device_bytes", "tbs_grid_harmonic_frequency", "tbs_set_concurrency", "tbs_set_launch_overlap", "tbs_last_error",
    "tbs_set_abl", "tbs_set_scheme", "tbs_set_boundary", "tbs_set_criterion", "tbs_set_kspace_absorption", "tbs_set_kspace_scatterer", "tbs_set_medium", "tbs_set_medium_host", "tbs_set_potential", "tbs_set_source",
    "tbs_set_source_field", "tbs_solve", "tbs_solve_host", "tbs_solve_resume", "tbs_solve_second_harmonic", "tbs_solve_harmonics",
    "tbs_apply_green", "tbs_get_potential", "tbs_get_source", "tbs_green_spectrum",
    "tbs_last_launch_count", "tbs_last_loop_ms", "tbs_profile_term", "tbs_set_graph_batch",
]

_lib = None


def load() -> ctypes.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} not found: the CUDA library is the only implementation of this package. "
            "Build it with `python -m paper_2507_13754_b200.build`.")
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double
    ip = ctypes.POINTER(ctypes.c_int32)
    dp = ctypes.POINTER(ctypes.c_double)
    fp = ctypes.POINTER(ctypes.c_float)
    L.tbs_version.restype = ctypes.c_char_p
    L.tbs_plan_create.argtypes = [ctypes.POINTER(vp), i32, ip, dbl, i32, dp, dbl, dbl]
    L.tbs_plan_destroy.argtypes = [vp]
    L.tbs_plan_destroy.restype = None
    L.tbs_plan_workspace_bytes.argtypes = [vp]
    L.tbs_plan_workspace_bytes.restype = ctypes.c_size_t
    L.tbs_plan_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    L.tbs_plan_device_bytes.argtypes = [vp]
    L.tbs_plan_device_bytes.restype = ctypes.c_size_t
    L.tbs_grid_harmonic_frequency.argtypes = [i32, dbl, i32, dbl]
    L.tbs_grid_harmonic_frequency.restype = dbl
    L.tbs_set_concurrency.argtypes = [vp, i32]
    L.tbs_set_launch_overlap.argtypes = [vp, i32]
    L.tbs_last_error.argtypes = [vp]
    L.tbs_last_error.restype = ctypes.c_char_p
    L.tbs_set_abl.argtypes = [vp, i32, dbl]
    L.tbs_set_scheme.argtypes = [vp, i32]
    L.tbs_set_boundary.argtypes = [vp, i32]
    L.tbs_set_kspace_absorption.argtypes = [vp, dbl, dbl, i32]
    L.tbs_set_kspace_scatterer.argtypes = [vp, vp, vp]
    L.tbs_set_criterion.argtypes = [vp, i32, i32]
    L.tbs_set_medium.argtypes = [vp, vp, vp, vp, dbl, dbl, dbl, dbl, vp]
    L.tbs_set_medium_host.argtypes = [vp, vp, vp, vp, dbl, dbl, dbl, dbl, vp]
    L.tbs_set_potential.argtypes = [vp, i32, vp, vp]
    L.tbs_set_source.argtypes = [vp, i32, dp, fp, vp]
    L.tbs_set_source_field.argtypes = [vp, i32, vp, vp]
    L.tbs_solve.argtypes = [vp, i32, dbl, vp, dp, ip, vp]
    L.tbs_solve_host.argtypes = [vp, i32, dbl, vp, dp, ip, vp]
    L.tbs_solve_resume.argtypes = [vp, i32, dbl, vp, dp, ip, vp]
    L.tbs_solve_second_harmonic.argtypes = [vp, vp, i32, dbl, i32, dbl, vp, vp, dp, dp, ip, ip, vp]
    L.tbs_solve_harmonics.argtypes = [ctypes.POINTER(vp), i32, i32, dbl, i32, dbl, ctypes.POINTER(vp),
                                      ctypes.POINTER(dp), ip, vp]
    L.tbs_apply_green.argtypes = [vp, i32, vp, vp, vp]
    L.tbs_get_potential.argtypes = [vp, i32, vp, vp]
    L.tbs_get_source.argtypes = [vp, i32, vp, vp]
    L.tbs_green_spectrum.argtypes = [vp, i32, vp, vp]
    L.tbs_last_launch_count.argtypes = [vp]
    L.tbs_last_launch_count.restype = i64
    L.tbs_last_loop_ms.argtypes = [vp]
    L.tbs_last_loop_ms.restype = dbl
    L.tbs_profile_term.argtypes = [vp, i32, i32, dp, vp]
    L.tbs_set_graph_batch.argtypes = [vp, i32]
    for name in SYMBOLS:
        fn = getattr(L, name)
        if fn.restype is ctypes.c_int and name not in ("tbs_version",):
            fn.restype = ctypes.c_int
    _lib = L
    return L
