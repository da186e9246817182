"""Exact-arithmetic gamma of single voxels (test helper; no floating point until the final square root).

Eq. 1 on the Kuhn-split piecewise-linear evaluation surface, evaluated with Python Fractions:
for every in-grid cell whose spatial lower bound is below the running minimum, every Kuhn simplex, every non-empty
subset of its vertices: the affine projection of the reference point by the normal equations,
accepted when all weights are >= 0.  The closest point of a simplex lies in the relative interior of one of its
faces, where that projection has positive weights, so the minimum over the accepted subsets is the exact distance.

Why it exists: under the LOCAL criterion a reference dose that is tiny against the evaluation doses around it
(D_r = 1e-10 Gy in the tail of the analytic beam phantom, dD_v = DD * D_r) stretches the dose axis by 1e10 and more;
the Gram matrix of the normal equations then has a condition number near 1e20 and the double-precision oracles
lose all digits there (the two oracles, Cholesky and Gaussian elimination, disagree by 0.4 on such voxels).  This
module says what gamma really is on a handful of them.  The inputs are the same fp32 numbers the boundary receives,
converted exactly.  Slow: seconds per voxel; small grids only.
"""
from fractions import Fraction
from itertools import combinations, permutations, product
import math

import numpy as np


def _solve(A, b):
    """Gaussian elimination over Fractions; None if singular."""
    n = len(b)
    M = [row[:] + [b[i]] for i, row in enumerate(A)]
    for c in range(n):
        p = next((r for r in range(c, n) if M[r][c] != 0), None)
        if p is None:
            return None
        M[c], M[p] = M[p], M[c]
        inv = 1 / M[c][c]
        for r in range(c + 1, n):
            if M[r][c] != 0:
                f = M[r][c] * inv
                for k in range(c, n + 1):
                    M[r][k] -= f * M[c][k]
    x = [Fraction(0)] * n
    for r in range(n - 1, -1, -1):
        x[r] = (M[r][n] - sum(M[r][k] * x[k] for k in range(r + 1, n))) / M[r][r]
    return x


def simplex_dist2(points):
    """Exact squared distance from the origin to conv(points); points: list of equal-length lists of Fractions."""
    best = None
    K = len(points[0])
    for size in range(1, len(points) + 1):
        for sub in combinations(points, size):
            base = sub[0]
            W = [[p[a] - base[a] for a in range(K)] for p in sub[1:]]
            if W:
                G = [[sum(u[a] * w[a] for a in range(K)) for w in W] for u in W]
                rhs = [-sum(u[a] * base[a] for a in range(K)) for u in W]
                lam = _solve(G, rhs)
                if lam is None or any(l < 0 for l in lam) or sum(lam) > 1:
                    continue
                foot = [base[a] + sum(l * w[a] for l, w in zip(lam, W)) for a in range(K)]
            else:
                foot = base
            d2 = sum(c * c for c in foot)
            if best is None or d2 < best:
                best = d2
    return best


def exact_gamma(ref, ev, dims, spacing_mm, dd, dta_mm, mode, voxel, norm_dose=None, gamma_ub=None):
    """gamma of the voxel with linear index `voxel` (x fastest); ref / ev: fp32 arrays; dd, dta_mm, spacing_mm: the
    fp32-rounded values; returns a float (sqrt of the exact minimum).  Excluded voxels are the caller's business.
    gamma_ub: a known upper bound of the result (it limits the cells that are enumerated when gamma_0 is astronomically
    large); the result is checked against it, so a wrong bound fails loudly instead of truncating the search."""
    ref = np.asarray(ref, dtype=np.float32).ravel()
    ev = np.asarray(ev, dtype=np.float32).ravel()
    F = lambda x: Fraction(float(np.float32(x)))  # noqa: E731  (a float converts exactly)
    axes = [a for a in range(3) if dims[a] > 1]
    n = len(axes)
    stride = [1, dims[0], dims[0] * dims[1]]
    v = [voxel % dims[0], (voxel // dims[0]) % dims[1], voxel // (dims[0] * dims[1])]
    h = [F(spacing_mm[a]) / F(dta_mm) for a in range(3)]
    Dr = F(ref[voxel])
    dnorm = F(ref.max()) if norm_dose is None else F(norm_dose)
    dD = F(dd) * (dnorm if mode == 0 else Dr)
    assert dD > 0
    best = ((F(ev[voxel]) - Dr) / dD) ** 2                       # gamma_0^2: the vertex at the voxel itself
    perms = list(permutations(range(n)))
    radius = math.sqrt(float(best)) if gamma_ub is None else min(math.sqrt(float(best)), float(gamma_ub))
    reach = [int(math.ceil(radius / float(h[a]))) + 1 for a in axes]
    cells = []
    for o in product(*[range(-r - 1, r + 1) for r in reach]):
        if any(not (0 <= v[axes[i]] + o[i] <= dims[axes[i]] - 2) for i in range(n)):
            continue
        b2 = sum((max(o[i], -o[i] - 1, 0) * h[axes[i]]) ** 2 for i in range(n))
        cells.append((b2, o))
    cells.sort()
    for b2, o in cells:
        if b2 >= best:
            break
        for pm in perms:
            u = [o[i] for i in range(n)]
            pts = []
            for m in range(n + 1):
                if m > 0:
                    u[pm[m - 1]] += 1
                lin = sum((v[axes[i]] + u[i]) * stride[axes[i]] for i in range(n)) + \
                    sum(v[a] * stride[a] for a in range(3) if a not in axes)
                pts.append([u[i] * h[axes[i]] for i in range(n)] + [(F(ev[lin]) - Dr) / dD])
            d2 = simplex_dist2(pts)
            if d2 < best:
                best = d2
    g = math.sqrt(float(best))
    assert gamma_ub is None or g <= gamma_ub, "gamma_ub was not an upper bound: the enumeration may have been cut short"
    return g
