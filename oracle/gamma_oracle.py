"""ctypes front end of oracle/gamma_oracle.c -- TEST INFRASTRUCTURE, not the product.

The arithmetic lives in gamma_oracle.c (double precision, written from
PAPER.md:149-209; see that file's header for citations and pins).  This module
only compiles it with gcc, widens the fp32 inputs to float64 exactly, and
marshals arguments.  It shares nothing with the CUDA path.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gamma_oracle.c")
_LIB = os.path.join(_HERE, "libgamma_oracle.so")
_lib = None

FORM_PLAIN, FORM_SHELL, FORM_VERTEX_ONLY = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile gamma_oracle.c -> libgamma_oracle.so (gcc -O2 -fopenmp, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_gamma.restype = ctypes.c_int
        lib.oracle_gamma.argtypes = [
            c_dp, c_dp, ctypes.POINTER(ctypes.c_int), c_dp,
            ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int,
            ctypes.POINTER(ctypes.c_longlong), ctypes.c_longlong, c_dp, ctypes.POINTER(ctypes.c_longlong),
            ctypes.c_int,
        ]
        for f in (lib.oracle_simplex_distance, lib.oracle_simplex_distance_ju):
            f.restype = ctypes.c_double
            f.argtypes = [c_dp, ctypes.c_int, ctypes.c_int]
        lib.oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def gamma(ref, ev, dims, spacing_mm, dd, dta_mm, mode=0, cutoff=0.1, norm_dose=0.0, form="shell",
          voxels=None, return_visits=False, nthreads=0):
    """gamma index of `ref` against `ev` (see oracle_gamma in gamma_oracle.c).

    `ref`, `ev`: arrays with nx*ny*nz elements, x fastest (any shape; flattened in C order).
    `dd`, `dta_mm`, `spacing_mm`, `cutoff`: pass the float32-rounded values the CUDA
    boundary receives if a bit-for-bit identical problem statement is wanted.
    Returns float64 gamma (NaN for excluded voxels): N values, or len(voxels) values.
    """
    lib = _load()
    r = np.ascontiguousarray(np.asarray(ref, dtype=np.float64).ravel())
    e = np.ascontiguousarray(np.asarray(ev, dtype=np.float64).ravel())
    nx, ny, nz = (int(d) for d in dims)
    if r.size != nx * ny * nz or e.size != r.size:
        raise ValueError("ref/eval size does not match dims")
    cdims = (ctypes.c_int * 3)(nx, ny, nz)
    sp = np.asarray(spacing_mm, dtype=np.float64).copy()
    f = {"plain": FORM_PLAIN, "shell": FORM_SHELL, "vertex": FORM_VERTEX_ONLY}[form]
    if voxels is None:
        vl, nl, count = None, 0, r.size
    else:
        vox = np.ascontiguousarray(np.asarray(voxels, dtype=np.int64).ravel())
        vl, nl, count = vox.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)), vox.size, vox.size
    out = np.empty(count, dtype=np.float64)
    vis = np.zeros(count, dtype=np.int64) if return_visits else None
    rc = lib.oracle_gamma(_dp(r), _dp(e), cdims, _dp(sp), float(dd), float(dta_mm), int(mode),
                          float(cutoff), float(norm_dose), f, vl, nl, _dp(out),
                          vis.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)) if return_visits else None,
                          int(nthreads))
    if rc != 0:
        raise ValueError("oracle_gamma: invalid arguments")
    return (out, vis) if return_visits else out


def simplex_distance(points) -> float:
    """Distance from the origin to conv(points); points: (nv, K) array.  All-subsets form."""
    q = np.ascontiguousarray(np.asarray(points, dtype=np.float64))
    return float(_load().oracle_simplex_distance(_dp(q), q.shape[0], q.shape[1]))


def simplex_distance_ju(points) -> float:
    """Same distance by the negative-weight recursion."""
    q = np.ascontiguousarray(np.asarray(points, dtype=np.float64))
    return float(_load().oracle_simplex_distance_ju(_dp(q), q.shape[0], q.shape[1]))
