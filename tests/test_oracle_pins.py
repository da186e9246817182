"""Pins for the CPU oracle (oracle/gamma_oracle.c): each test checks it against
something OTHER than itself -- a closed form, an invariant of Eq. 1, a textbook
special case, a library optimiser or brute force -- chosen so that a dropped
term, a wrong sign/index or a transposed operand fails at least one of them.

Citations are PAPER.md lines (arxiv/paper_1012_1900).  None of these tests needs a GPU.
"""
import itertools
import os

import numpy as np
import pytest
from scipy.optimize import minimize

HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------
# independent helpers (no oracle code)
# ----------------------------------------------------------------------------
def kuhn_simplices_of_cell(c, n):
    """Vertex chains c, c+e_p1, c+e_p1+e_p2, ... for every permutation p."""
    out = []
    for perm in itertools.permutations(range(n)):
        v = np.array(c, dtype=np.int64)
        chain = [v.copy()]
        for a in perm:
            v = v.copy()
            v[a] += 1
            chain.append(v)
        out.append(np.array(chain))
    return out


def all_simplex_points(ev, v, spacing, dta, Dr, dD):
    """All Kuhn simplices of the grid `ev` (indexed [x,y,(z)]) as arrays of points in the
    normalised dose-distance space relative to the reference point of voxel v."""
    n = ev.ndim
    simp = []
    for c in itertools.product(*[range(s - 1) for s in ev.shape]):
        for chain in kuhn_simplices_of_cell(c, n):
            pts = np.zeros((n + 1, n + 1))
            for i, u in enumerate(chain):
                pts[i, :n] = (u - np.array(v)) * np.array(spacing[:n]) / dta
                pts[i, n] = (ev[tuple(u)] - Dr) / dD
            simp.append(pts)
    return simp


def qp_simplex_distance(pts):
    """min |sum w_i p_i| over the probability simplex, by a library optimiser (SLSQP)."""
    k = pts.shape[0]
    best = np.inf
    for start in list(np.eye(k)) + [np.full(k, 1.0 / k)]:
        res = minimize(lambda w: float(np.sum((w @ pts) ** 2)), start, jac=lambda w: 2 * pts @ (w @ pts),
                       bounds=[(0, 1)] * k, constraints=[{"type": "eq", "fun": lambda w: np.sum(w) - 1.0,
                                                          "jac": lambda w: np.ones(k)}],
                       method="SLSQP", options={"ftol": 1e-16, "maxiter": 500})
        best = min(best, float(np.sqrt(max(res.fun, 0.0))))
    return best


def to_xyz_order(a):
    """phantoms / the C layout are [z,y,x]; helper tests index [x,y,z]."""
    return np.transpose(a, tuple(range(a.ndim))[::-1])


def run_oracle(oracle_mod, ref_zyx, ev_zyx, spacing, dd, dta, **kw):
    nz, ny, nx = ref_zyx.shape
    out = oracle_mod.gamma(ref_zyx, ev_zyx, (nx, ny, nz), spacing, dd, dta, **kw)
    return out.reshape(ref_zyx.shape) if kw.get("voxels") is None else out


# ----------------------------------------------------------------------------
# point-to-simplex routine
# ----------------------------------------------------------------------------
def test_simplex_distance_textbook_cases(oracle_mod):
    d = oracle_mod.simplex_distance
    # single vertex
    assert d([[3.0, 4.0]]) == pytest.approx(5.0, abs=1e-15)
    # segment, interior foot: segment from (1,-1) to (1,2): closest point (1,0)
    assert d([[1.0, -1.0], [1.0, 2.0]]) == pytest.approx(1.0, abs=1e-15)
    # segment, foot beyond an end -> end vertex
    assert d([[1.0, 1.0], [1.0, 2.0]]) == pytest.approx(np.sqrt(2.0), abs=1e-15)
    # triangle in R^3 in the plane z = 2, origin projects inside
    assert d([[-1, -1, 2.0], [3, -1, 2.0], [-1, 3, 2.0]]) == pytest.approx(2.0, abs=1e-14)
    # same triangle moved so that the projection falls beyond the edge x = 1
    assert d([[1, -1, 2.0], [5, -1, 2.0], [1, 3, 2.0]]) == pytest.approx(np.sqrt(1 + 4), abs=1e-14)
    # beyond a corner
    assert d([[1, 1, 2.0], [5, 1, 2.0], [1, 5, 2.0]]) == pytest.approx(np.sqrt(1 + 1 + 4), abs=1e-14)
    # tetrahedron in R^4 lying in the hyperplane w = 3 and containing the projection
    tet = [[-1, -1, -1, 3.0], [4, -1, -1, 3.0], [-1, 4, -1, 3.0], [-1, -1, 4, 3.0]]
    assert d(tet) == pytest.approx(3.0, abs=1e-14)


@pytest.mark.parametrize("K,nv", [(2, 2), (3, 2), (3, 3), (4, 2), (4, 3), (4, 4)])
def test_all_subsets_equals_ju_recursion_and_library_qp(oracle_mod, K, nv):
    """Two algorithms of the paper (PAPER.md:256 vs 209) and a library QP agree; random
    barycentric sampling never finds a closer point."""
    rng = np.random.default_rng([7, K, nv])
    for trial in range(60):
        pts = rng.normal(size=(nv, K)) * rng.uniform(0.2, 3.0)
        pts += rng.normal(size=(1, K)) * rng.uniform(0.0, 2.0)
        a = oracle_mod.simplex_distance(pts)
        b = oracle_mod.simplex_distance_ju(pts)
        assert a == pytest.approx(b, abs=1e-12)
        assert a == pytest.approx(qp_simplex_distance(pts), abs=2e-7)
        w = rng.dirichlet(np.full(nv, 0.5), size=4000)
        assert np.min(np.linalg.norm(w @ pts, axis=1)) >= a - 1e-12


# ----------------------------------------------------------------------------
# whole pipeline: invariants of Eq. 1
# ----------------------------------------------------------------------------
def test_identical_grids_give_zero(oracle_mod):
    rng = np.random.default_rng(1)
    ref = rng.uniform(0.5, 2.0, size=(5, 6, 7))
    g = run_oracle(oracle_mod, ref, ref, (2.0, 3.0, 2.5), 0.03, 3.0, cutoff=0.0)
    assert np.all(g == 0.0)


@pytest.mark.parametrize("shape", [(1, 6, 7), (4, 5, 6)])
def test_flat_fields_uniform_offset(oracle_mod, shape):
    """Flat D_r = a, D_e = a + c: the surface is the plane D = a + c, gamma = |c|/dD."""
    a, c, dd = 1.7, -0.08, 0.03
    ref = np.full(shape, a)
    ev = np.full(shape, a + c)
    for form in ("plain", "shell"):
        g = run_oracle(oracle_mod, ref, ev, (2.0, 2.5, 3.0), dd, 3.0, cutoff=0.0, form=form)
        assert np.allclose(g, abs(c) / (dd * a), rtol=0, atol=1e-13)


def test_gamma_never_exceeds_gamma0_and_vertex_only(oracle_mod):
    rng = np.random.default_rng(3)
    ref = rng.uniform(0.8, 2.0, size=(6, 7, 8))
    ev = ref * 1.03 + rng.normal(0, 0.05, size=ref.shape)
    sp, dd, dta = (2.0, 2.5, 3.0), 0.03, 3.0
    g = run_oracle(oracle_mod, ref, ev, sp, dd, dta, cutoff=0.0)
    gv = run_oracle(oracle_mod, ref, ev, sp, dd, dta, cutoff=0.0, form="vertex")
    g0 = np.abs(ev - ref) / (dd * ref.max())
    assert np.all(g <= g0 + 1e-15)
    assert np.all(g <= gv + 1e-15)          # interpolation can only lower gamma
    assert np.any(g < gv - 1e-6)            # ... and does, somewhere


def _load_golden():
    vals = {}
    with open(os.path.join(HERE, "golden", "ramp_closed_form.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            vals[k] = [float(x) for x in v]
    return vals


def test_ramp_closed_form_golden_3d(oracle_mod):
    """Linear ramp, sub-voxel shift: gamma = |g.s| / sqrt(dD^2 + dd^2 |g|^2)."""
    G = _load_golden()
    n = int(G["n"][0])
    h = G["spacing_mm"]
    g = np.array(G["gradient_Gy_per_mm"])
    s = np.array(G["shift_mm"])
    dD, dta = G["delta_D_Gy"][0], G["dta_mm"][0]
    ax = [(np.arange(n) - (n - 1) / 2) * hh for hh in h]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    ref = G["offset_Gy"][0] + g[0] * X + g[1] * Y + g[2] * Z
    ev = G["offset_Gy"][0] + g[0] * (X - s[0]) + g[1] * (Y - s[1]) + g[2] * (Z - s[2])
    closed = abs(g @ s) / np.sqrt(dD ** 2 + dta ** 2 * (g @ g))
    assert closed == pytest.approx(G["expected_gamma"][0], abs=1e-12)
    for form in ("plain", "shell"):
        out = run_oracle(oracle_mod, ref, ev, h, dD, dta, cutoff=0.0, norm_dose=1.0, form=form)
        assert out[n // 2, n // 2, n // 2] == pytest.approx(G["expected_gamma"][0], abs=1e-12)
        # interior voxels (farther than gamma*dta + one voxel from the border) all agree
        assert np.allclose(out[2:-2, 2:-2, 2:-2], closed, rtol=0, atol=1e-12)
        out2 = run_oracle(oracle_mod, ref, ev, h, 2 * dD, 2 * dta, cutoff=0.0, norm_dose=1.0, form=form)
        assert out2[n // 2, n // 2, n // 2] == pytest.approx(G["expected_gamma_doubled_criteria"][0], abs=1e-12)


def test_ramp_closed_form_2d_anisotropic(oracle_mod):
    nx, ny = 11, 9
    h = (2.0, 3.5, 1.0)
    g = np.array([0.03, 0.045])
    x = (np.arange(nx) - (nx - 1) / 2) * h[0]
    y = (np.arange(ny) - (ny - 1) / 2) * h[1]
    Y, X = np.meshgrid(y, x, indexing="ij")
    ref = (5.0 + g[0] * X + g[1] * Y)[None]
    ev = ref + 0.04                      # D_r - D_e(x_r) = -0.04 everywhere
    dD, dta = 0.05, 2.0
    closed = 0.04 / np.sqrt(dD ** 2 + dta ** 2 * (g @ g))
    out = run_oracle(oracle_mod, ref, ev, h, dD, dta, cutoff=0.0, norm_dose=1.0)
    assert np.allclose(out[0, 2:-2, 2:-2], closed, rtol=0, atol=1e-12)


def test_criteria_scaling_law_and_monotonicity(oracle_mod):
    """gamma(k dD, k dd) = gamma(dD, dd)/k exactly; non-increasing in dD alone and in dd
    alone (phenomena 1-3)."""
    rng = np.random.default_rng(11)
    ref = rng.uniform(0.8, 2.0, size=(5, 6, 7))
    ev = ref * 0.98 + rng.normal(0, 0.04, size=ref.shape)
    sp = (2.0, 2.5, 3.0)
    base = run_oracle(oracle_mod, ref, ev, sp, 0.02, 2.0, cutoff=0.0)
    for k in (2.0, 3.0):
        scaled = run_oracle(oracle_mod, ref, ev, sp, 0.02 * k, 2.0 * k, cutoff=0.0)
        assert np.allclose(scaled * k, base, rtol=1e-12, atol=1e-13)
    more_dd = run_oracle(oracle_mod, ref, ev, sp, 0.03, 2.0, cutoff=0.0)
    more_dta = run_oracle(oracle_mod, ref, ev, sp, 0.02, 3.0, cutoff=0.0)
    assert np.all(more_dd <= base + 1e-13)
    assert np.all(more_dta <= base + 1e-13)


def test_axis_permutation_invariance(oracle_mod):
    """The Kuhn split is invariant under permutations of the axes (with their spacings)."""
    rng = np.random.default_rng(13)
    ref = rng.uniform(0.8, 2.0, size=(4, 5, 6))      # [z,y,x]
    ev = ref * 1.02 + rng.normal(0, 0.05, size=ref.shape)
    sp = np.array([2.0, 2.5, 3.0])                   # (dx,dy,dz)
    base = run_oracle(oracle_mod, ref, ev, sp, 0.03, 2.5, cutoff=0.0)
    for perm in itertools.permutations(range(3)):
        # array axes are (z,y,x) = reversed spatial axes
        arr_perm = tuple(2 - perm[2 - i] for i in range(3))
        r2 = np.ascontiguousarray(np.transpose(ref, arr_perm))
        e2 = np.ascontiguousarray(np.transpose(ev, arr_perm))
        sp2 = sp[list(perm)]
        g2 = run_oracle(oracle_mod, r2, e2, sp2, 0.03, 2.5, cutoff=0.0)
        assert np.allclose(np.transpose(base, arr_perm), g2, rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------
# brute force on tiny grids
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("shape,spacing,dd,dta", [
    ((3, 3, 3), (2.0, 2.5, 3.0), 0.03, 3.0),
    ((2, 3, 4), (3.0, 1.5, 2.0), 0.05, 1.5),
    ((4, 4), (2.5, 2.0, 1.0), 0.03, 2.0),
    ((3, 5), (1.0, 2.0, 1.0), 0.02, 3.0),
])
def test_bruteforce_all_simplices_library_qp_and_sampling(oracle_mod, shape, spacing, dd, dta):
    """gamma[v] == min over ALL simplices of the grid (no search radius, no pruning) of a
    library-QP distance; dense barycentric sampling approaches it from above."""
    rng = np.random.default_rng([17, len(shape), shape[0]])
    n = len(shape)
    ref_xyz = rng.uniform(0.9, 2.0, size=shape)
    ev_xyz = ref_xyz * rng.uniform(0.95, 1.05) + rng.normal(0, 0.06, size=shape)
    ref = to_xyz_order(ref_xyz)[None] if n == 2 else to_xyz_order(ref_xyz)
    ev = to_xyz_order(ev_xyz)[None] if n == 2 else to_xyz_order(ev_xyz)
    dnorm = ref.max()
    out = run_oracle(oracle_mod, ref, ev, spacing, dd, dta, cutoff=0.0)
    out_xyz = to_xyz_order(out[0] if n == 2 else out)
    dD = dd * dnorm
    for v in itertools.product(*[range(s) for s in shape]):
        Dr = ref_xyz[v]
        simp = all_simplex_points(ev_xyz, v, spacing, dta, Dr, dD)
        exact = min(qp_simplex_distance(p) for p in simp)
        assert out_xyz[v] == pytest.approx(exact, abs=5e-7)
        # brute force: coarse Dirichlet sampling of every simplex, then shrinking random
        # perturbations around the best samples of the few most promising simplices
        w = rng.dirichlet(np.full(n + 1, 0.6), size=600)
        coarse = []
        for p in simp:
            dist = np.linalg.norm(w @ p, axis=1)
            j = int(np.argmin(dist))
            coarse.append((dist[j], w[j]))
        sampled = min(c[0] for c in coarse)
        for si in np.argsort([c[0] for c in coarse])[:6]:
            best_d, best_w = coarse[si]
            for r in (0.3, 0.1, 0.03, 0.01, 0.003, 0.001):
                cand = np.clip(best_w[None, :] + r * rng.normal(size=(400, n + 1)), 0.0, None)
                cand = cand[cand.sum(axis=1) > 0]
                cand /= cand.sum(axis=1, keepdims=True)
                dist = np.linalg.norm(cand @ simp[si], axis=1)
                j = int(np.argmin(dist))
                if dist[j] < best_d:
                    best_d, best_w = dist[j], cand[j]
            sampled = min(sampled, best_d)
        assert sampled >= out_xyz[v] - 1e-12
        assert sampled <= out_xyz[v] + 5e-3


def test_one_d_polyline_by_hand(oracle_mod):
    """n = 1: the surface is a polyline; distance to each segment by the clamped-foot
    formula.  A 2D grid whose dose does not depend on y gives the same gamma."""
    rng = np.random.default_rng(19)
    nx, h, dd, dta = 12, 2.0, 0.03, 2.5
    ref1 = rng.uniform(0.9, 2.0, size=nx)
    ev1 = ref1 * 1.04 + rng.normal(0, 0.08, size=nx)
    dD = dd * ref1.max()
    expect = np.empty(nx)
    for i in range(nx):
        best = np.inf
        for j in range(nx - 1):
            p0 = np.array([(j - i) * h / dta, (ev1[j] - ref1[i]) / dD])
            p1 = np.array([(j + 1 - i) * h / dta, (ev1[j + 1] - ref1[i]) / dD])
            e = p1 - p0
            t = np.clip(-(p0 @ e) / (e @ e), 0.0, 1.0)
            best = min(best, np.linalg.norm(p0 + t * e))
        expect[i] = best
    out1 = oracle_mod.gamma(ref1, ev1, (nx, 1, 1), (h, 1.0, 1.0), dd, dta, cutoff=0.0)
    assert np.allclose(out1, expect, rtol=0, atol=1e-12)
    ny = 9
    ref2 = np.tile(ref1, (1, ny, 1))
    ev2 = np.tile(ev1, (1, ny, 1))
    out2 = oracle_mod.gamma(ref2, ev2, (nx, ny, 1), (h, 3.0, 1.0), dd, dta, cutoff=0.0).reshape(ny, nx)
    assert np.allclose(out2, expect[None, :], rtol=0, atol=1e-12)


def _kuhn_interp(ev_xyz, pts):
    """Evaluate the Kuhn piecewise-linear interpolant of ev_xyz at fractional index points."""
    n = ev_xyz.ndim
    out = np.empty(len(pts))
    for i, p in enumerate(pts):
        c = np.minimum(np.floor(p).astype(int), np.array(ev_xyz.shape) - 2)
        f = p - c
        order = np.argsort(-f, kind="stable")
        v = c.copy()
        val = ev_xyz[tuple(v)] * (1 - f[order[0]])
        for m in range(n):
            v = v.copy()
            v[order[m]] += 1
            wgt = f[order[m]] - (f[order[m + 1]] if m + 1 < n else 0.0)
            val += ev_xyz[tuple(v)] * wgt
        out[i] = val
    return out


def test_vertex_only_on_refined_kuhn_interpolant_converges_from_above(oracle_mod):
    rng = np.random.default_rng(23)
    shape = (6, 6)
    spacing = (2.5, 2.5, 1.0)
    # gentle field: the vertex-only error is about half the refined step measured in the
    # normalised space, so neighbouring doses must not differ by many dD
    ref_xyz = rng.uniform(1.50, 1.56, size=shape)
    ev_xyz = ref_xyz * 1.02 + rng.normal(0, 0.005, size=shape)
    dd, dta = 0.03, 3.0
    dnorm = ref_xyz.max()
    gi = oracle_mod.gamma(to_xyz_order(ref_xyz), to_xyz_order(ev_xyz), (6, 6, 1), spacing, dd, dta,
                          cutoff=0.0).reshape(6, 6).T
    gaps = []
    for k in (2, 16):
        m = (shape[0] - 1) * k + 1
        idx = np.arange(m) / k
        P = np.array([(a, b) for a in idx for b in idx])
        fine = _kuhn_interp(ev_xyz, P).reshape(m, m)
        ref_fine = np.zeros((m, m))
        ref_fine[::k, ::k] = ref_xyz
        gv = oracle_mod.gamma(to_xyz_order(ref_fine), to_xyz_order(fine), (m, m, 1),
                              (spacing[0] / k, spacing[1] / k, 1.0), dd, dta, cutoff=0.0,
                              norm_dose=dnorm, form="vertex").reshape(m, m).T[::k, ::k]
        assert np.all(gv >= gi - 1e-12)
        gaps.append(np.max(gv - gi))
    assert gaps[1] < gaps[0]
    assert gaps[1] < 0.03


# ----------------------------------------------------------------------------
# search-region handling
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("case", ["cfg1", "cfg2_small"])
def test_plain_radius_equals_shell_form(oracle_mod, case):
    from paper_1012_1900_b200.phantoms import make_case

    c = make_case(case)
    a = oracle_mod.gamma(c.ref, c.eval, c.dims, c.spacing_mm, c.dd, c.dta_mm, c.mode, c.cutoff, form="plain")
    b = oracle_mod.gamma(c.ref, c.eval, c.dims, c.spacing_mm, c.dd, c.dta_mm, c.mode, c.cutoff, form="shell")
    assert np.array_equal(np.isnan(a), np.isnan(b))
    m = ~np.isnan(a)
    assert m.sum() > 100
    assert np.array_equal(a[m], b[m])       # bit for bit


def test_large_dose_difference_needs_unbounded_radius(oracle_mod):
    """no fixed search radius.  One far-away matching voxel must be found."""
    nx = 40
    ref = np.full((1, 3, nx), 1.0)
    ev = np.full((1, 3, nx), 3.0)
    ev[:, :, 30:] = 1.0                      # exact agreement 25 voxels away from voxel 5
    out = oracle_mod.gamma(ref, ev, (nx, 3, 1), (1.0, 1.0, 1.0), 0.03, 1.0, cutoff=0.0).reshape(3, nx)
    # gamma0 = 2/0.03 = 66.7.  Between x = 29 and x = 30 the interpolant is the straight
    # segment (24, s) -> (25, 0) with s = 2/0.03 in normalised units; the foot of the
    # perpendicular from the origin lies inside it: distance = 25 s / sqrt(1 + s^2)
    s = 2.0 / 0.03
    assert out[1, 5] == pytest.approx(25.0 * s / np.sqrt(1.0 + s * s), abs=1e-11)
    assert 24.99 < out[1, 5] < 25.0
    assert out[1, 35] == 0.0


def test_visit_counts_scale_as_gamma_cubed(oracle_mod):
    """N_s(v) = #cells with L_cell < gamma grows like gamma^n."""
    ref = np.full((41, 41, 41), 1.0)
    counts = []
    for c in (0.15, 0.30):
        ev = ref + c
        g, vis = oracle_mod.gamma(ref, ev, (41, 41, 41), (1.0, 1.0, 1.0), 0.03, 1.0, cutoff=0.0,
                                  voxels=[20 + 41 * (20 + 41 * 20)], return_visits=True)
        assert g[0] == pytest.approx(c / 0.03, abs=1e-12)
        counts.append(vis[0])
    assert 6.0 < counts[1] / counts[0] < 10.0      # (2x gamma)^3 = 8


@pytest.mark.parametrize("shape,spacing,dd,dta,mode", [
    ((3, 3, 3), (2.0, 2.5, 3.0), 0.03, 3.0, 0),
    ((5, 4, 6), (3.0, 1.5, 2.0), 0.02, 2.5, 0),
    ((7, 7, 7), (1.0, 1.0, 1.0), 0.01, 1.0, 1),        # deep: gamma_0 of several voxels, box clipped by the grid
    ((6, 9), (2.5, 2.0, 1.0), 0.03, 2.0, 0),
])
def test_vertex_only_form_equals_bruteforce_over_every_grid_vertex(oracle_mod, shape, spacing, dd, dta, mode):
    """The classical discrete gamma (Low et al.; the comparator of PAPER.md:135-137): the minimum of Gamma (Eq. 1,
    PAPER.md:149-162) over EVERY evaluation grid point, no radius, no pruning -- numpy over the whole grid."""
    rng = np.random.default_rng([31, len(shape), shape[0]])
    n = len(shape)
    ref_xyz = rng.uniform(0.9, 2.0, size=shape)
    ev_xyz = ref_xyz * rng.uniform(0.95, 1.05) + rng.normal(0, 0.08, size=shape)
    ref = to_xyz_order(ref_xyz)[None] if n == 2 else to_xyz_order(ref_xyz)
    ev = to_xyz_order(ev_xyz)[None] if n == 2 else to_xyz_order(ev_xyz)
    out = run_oracle(oracle_mod, ref, ev, spacing, dd, dta, mode=mode, cutoff=0.0, form="vertex")
    out_xyz = to_xyz_order(out[0] if n == 2 else out)
    idx = np.stack(np.meshgrid(*[np.arange(k) for k in shape], indexing="ij"), axis=-1).astype(np.float64)
    hn = np.array(spacing[:n]) / dta
    for v in itertools.product(*[range(k) for k in shape]):
        dD = dd * (ref_xyz.max() if mode == 0 else ref_xyz[v])
        spatial2 = (((idx - np.array(v, dtype=np.float64)) * hn) ** 2).sum(axis=-1)
        brute = np.sqrt(spatial2 + ((ev_xyz - ref_xyz[v]) / dD) ** 2).min()
        assert out_xyz[v] == pytest.approx(brute, abs=1e-12)


@pytest.mark.parametrize("shape,spacing,dd,dta", [
    ((7, 7, 7), (1.0, 1.0, 1.0), 0.02, 1.0),
    ((7, 6, 5), (2.0, 1.0, 1.5), 0.02, 1.5),
    ((8, 7), (1.0, 2.0, 1.0), 0.01, 1.5),
])
def test_visit_counts_equal_explicit_enumeration(oracle_mod, shape, spacing, dd, dta):
    """N_s(v) = #{in-grid cells c : L_cell(c - v) < gamma[v]} ("search length L ~ gamma"; DESIGN.md
    reading 4 for L_cell): counted here by a plain loop over every CELL of the grid, exact integers."""
    rng = np.random.default_rng([37, len(shape), shape[1]])
    n = len(shape)
    ref_xyz = rng.uniform(0.9, 2.0, size=shape)
    ev_xyz = ref_xyz * 1.03 + rng.normal(0, 0.10, size=shape)
    ref = to_xyz_order(ref_xyz)[None] if n == 2 else to_xyz_order(ref_xyz)
    ev = to_xyz_order(ev_xyz)[None] if n == 2 else to_xyz_order(ev_xyz)
    dims = tuple(shape) + (1,) * (3 - n)
    gam, vis = oracle_mod.gamma(ref, ev, dims, spacing, dd, dta, cutoff=0.0, return_visits=True)
    full = ref.shape if n == 3 else ref.shape[1:]
    gam_xyz, vis_xyz = to_xyz_order(gam.reshape(full)), to_xyz_order(vis.reshape(full))
    hn = [spacing[a] / dta for a in range(n)]
    total = 0
    for v in itertools.product(*[range(k) for k in shape]):
        cnt = 0
        for c in itertools.product(*[range(k - 1) for k in shape]):
            s = 0.0
            for a in range(n):
                o = c[a] - v[a]
                d = float(max(o, -o - 1, 0)) * hn[a]
                s += d * d
            cnt += np.sqrt(s) < gam_xyz[v]
        assert vis_xyz[v] == cnt, (v, vis_xyz[v], cnt)
        total += cnt
    assert total > 2 * np.prod(shape)            # the case is not trivial: more than the touching cells are counted


# ----------------------------------------------------------------------------
# conventions the paper does not pin (readings 8-12): checked as stated
# ----------------------------------------------------------------------------
def test_cutoff_local_mode_and_nan_policy(oracle_mod):
    rng = np.random.default_rng(29)
    ref = rng.uniform(0.0, 2.0, size=(4, 5, 6))
    ref[0, 0, 0] = 0.0
    ev = ref + 0.02
    sp = (2.0, 2.0, 2.0)
    g = run_oracle(oracle_mod, ref, ev, sp, 0.03, 3.0, cutoff=0.25)
    excl = ref < 0.25 * ref.max()
    assert np.array_equal(np.isnan(g), excl)
    # local mode: dD_v = DD * D_r[v]; D_r = 0 -> NaN even with cutoff 0
    gl = run_oracle(oracle_mod, ref, ev, sp, 0.03, 3.0, mode=1, cutoff=0.0)
    assert np.isnan(gl[0, 0, 0])
    # flat local: gamma = c / (DD * a)
    flat = np.full((3, 4, 5), 1.5)
    gl2 = run_oracle(oracle_mod, flat, flat + 0.03, sp, 0.03, 3.0, mode=1, cutoff=0.0)
    assert np.allclose(gl2, 0.03 / (0.03 * 1.5), atol=1e-13)
    # explicit normalisation dose
    gn = run_oracle(oracle_mod, flat, flat + 0.03, sp, 0.03, 3.0, cutoff=0.0, norm_dose=3.0)
    assert np.allclose(gn, 0.03 / (0.03 * 3.0), atol=1e-13)


def test_invalid_arguments_rejected(oracle_mod):
    a = np.ones((2, 2, 2))
    with pytest.raises(ValueError):
        oracle_mod.gamma(a, a, (2, 2, 2), (1, 1, 1), -0.03, 3.0)
    with pytest.raises(ValueError):
        oracle_mod.gamma(a, a, (2, 2, 2), (1, 1, 1), 0.03, 3.0, cutoff=1.0)
    with pytest.raises(ValueError):
        oracle_mod.gamma(a, a, (2, 2, 3), (1, 1, 1), 0.03, 3.0)
