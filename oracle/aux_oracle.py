"""Plain numpy definitions of the small steps around the gamma search -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It shares nothing with the CUDA path and never imports paper_1012_1900_b200.

  stats(gamma, nbins, hist_max)           pass rate / histogram / sums (BASELINE.json north_star (5); the paper
                                          only uses sum gamma^3 as its work predictor)
  sort_pairs(keys, vals, begin, end)      stable ascending sort of (key, value) on key bits [begin, end)
                                          (Algorithm A2 step 3: "sort {voxel index, DD}")
  offset_table(dims, spacing, dta, R)     Algorithm A1 steps 2-3 with the cell bound of
                                          DESIGN.md reading 4: the octant entries m >= 0 with L(m) < R, L^2 =
                                          sum_a (m_a h_a / dta)^2, sorted ascending by L

Pins (tests/test_aux_oracle_pins.py): hand-counted tiny inputs; the table sizes SURVEY.md section 8(a) lists
(full-space count = 8 x octant count in 3D); numpy's own stable sort on full keys.
"""
from __future__ import annotations

import numpy as np


def stats(gamma, nbins: int, hist_max: float):
    """Definition of gamma_stats: NaN = excluded; bin b counts finite gamma with floor(gamma / hist_max * nbins) == b,
    the last bin also takes everything >= hist_max.  The inputs are fp32 values (gamma, hist_max as the boundary receives
    it); the bin is the plain real-number definition evaluated in float64 -- no device rounding in it (DESIGN.md reading
    20: a kernel that decides the bin from an fp32 product may put a value that sits within an fp32 ulp of a bin edge
    into the neighbouring bin; the GPU tests allow exactly that and nothing else)."""
    g = np.asarray(gamma, dtype=np.float32).ravel()
    fin = ~np.isnan(g)
    gf = g[fin]
    g64 = gf.astype(np.float64)
    t = g64 * float(nbins) / float(np.float32(hist_max))
    b = np.minimum(np.floor(np.maximum(t, 0.0)), nbins - 1).astype(np.int64)
    hist = np.bincount(b, minlength=nbins).astype(np.int64)
    return hist, {
        "n_eval": int(fin.sum()),
        "n_pass": int((gf <= np.float32(1.0)).sum()),
        "sum_gamma": float(g64.sum()),
        "sum_gamma3": float((g64 ** 3).sum()),
        "max_gamma": float(gf.max()) if gf.size else 0.0,
        "n_nan": int((~fin).sum()),
    }


def sort_pairs(keys, vals, begin_bit: int = 0, end_bit: int = 32):
    """Stable ascending sort of (key, value) by the key bits [begin_bit, end_bit)."""
    k = np.asarray(keys).view(np.uint32).ravel()
    v = np.asarray(vals).view(np.uint32).ravel()
    width = end_bit - begin_bit
    digit = (k >> np.uint32(begin_bit)) & np.uint32((1 << width) - 1 if width < 32 else 0xFFFFFFFF)
    order = np.argsort(digit, kind="stable")
    return k[order], v[order]


def offset_table(dims, spacing_mm, dta_mm: float, radius: float):
    """Octant entries (m_x, m_y, m_z, L^2) with m_a in [0, dims_a - 1], L < radius, ascending in L.
    A dropped axis (size 1) has h = 0 and only m = 0."""
    h = [float(s) / float(dta_mm) if n > 1 else 0.0 for s, n in zip(spacing_mm, dims)]
    out = []
    lim = []
    for a in range(3):
        if h[a] > 0.0:
            lim.append(min(dims[a] - 1, int(np.floor(radius / h[a]))) + 1)
        else:
            lim.append(1)
    for mz in range(lim[2]):
        for my in range(lim[1]):
            for mx in range(lim[0]):
                L2 = (mx * h[0]) ** 2 + (my * h[1]) ** 2 + (mz * h[2]) ** 2
                if np.sqrt(L2) < radius:
                    out.append((L2, mx, my, mz))
    out.sort()
    return out
