"""ctypes front end of oracle/gamma_general_oracle.c -- TEST INFRASTRUCTURE, not the product.

The arithmetic lives in gamma_general_oracle.c (double precision, written from PAPER.md:149-162 and 204-207; see that
file's header for citations and pins): the gamma index with the evaluation dose on its own grid, plus the closest
point of the evaluation surface.  This module only compiles it with gcc, widens the fp32 inputs to float64 exactly
and marshals arguments.  It shares nothing with the CUDA path.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gamma_general_oracle.c")
_LIB = os.path.join(_HERE, "libgamma_general_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile gamma_general_oracle.c -> libgamma_general_oracle.so (gcc -O2 -fopenmp, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"], check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        lib.oracle_gamma_general.restype = ctypes.c_int
        lib.oracle_gamma_general.argtypes = [dp, ip, dp, dp, dp, ip, dp, dp, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                             ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                             ctypes.POINTER(ctypes.c_longlong), ctypes.c_longlong, dp, dp, ctypes.c_int]
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def gamma_general(ref, ref_dims, ref_spacing_mm, ref_origin_mm, ev, eval_dims, eval_spacing_mm, eval_origin_mm, dd, dta_mm,
                  mode=0, cutoff=0.1, norm_dose=0.0, form="shell", voxels=None, return_closest=False, nthreads=0):
    """gamma of `ref` (on its grid) against `ev` (on its own grid); see oracle_gamma_general in gamma_general_oracle.c.

    Arrays hold nx*ny*nz elements, x fastest (any shape; flattened in C order).  Returns float64 gamma (NaN = excluded),
    and with return_closest the (count, 4) array of closest points (x, y, z in mm, evaluation dose there).
    """
    lib = _load()
    r = np.ascontiguousarray(np.asarray(ref, dtype=np.float64).ravel())
    e = np.ascontiguousarray(np.asarray(ev, dtype=np.float64).ravel())
    rd = (ctypes.c_int * 3)(*[int(d) for d in ref_dims])
    ed = (ctypes.c_int * 3)(*[int(d) for d in eval_dims])
    if r.size != int(np.prod(ref_dims)) or e.size != int(np.prod(eval_dims)):
        raise ValueError("ref / eval size does not match dims")
    rs, ro = np.asarray(ref_spacing_mm, dtype=np.float64).copy(), np.asarray(ref_origin_mm, dtype=np.float64).copy()
    es, eo = np.asarray(eval_spacing_mm, dtype=np.float64).copy(), np.asarray(eval_origin_mm, dtype=np.float64).copy()
    if voxels is None:
        vl, nl, count = None, 0, r.size
    else:
        vox = np.ascontiguousarray(np.asarray(voxels, dtype=np.int64).ravel())
        vl, nl, count = vox.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)), vox.size, vox.size
    out = np.empty(count, dtype=np.float64)
    clo = np.empty((count, 4), dtype=np.float64) if return_closest else None
    rc = lib.oracle_gamma_general(_dp(r), rd, _dp(rs), _dp(ro), _dp(e), ed, _dp(es), _dp(eo), float(dd), float(dta_mm),
                                  int(mode), float(cutoff), float(norm_dose), {"all": 0, "shell": 1}[form], vl, nl, _dp(out),
                                  _dp(clo) if return_closest else None, int(nthreads))
    if rc != 0:
        raise ValueError("oracle_gamma_general: invalid arguments")
    return (out, clo) if return_closest else out
