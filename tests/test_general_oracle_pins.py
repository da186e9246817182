"""Pins for oracle/gamma_general_oracle.c (evaluation dose on its own grid + closest point):
each test checks it against something OTHER than itself -- the pinned same-grid oracle, a closed form, a library QP
over every simplex, an independent interpolator.  Citations are PAPER.md lines.  No GPU needed."""
import itertools

import numpy as np
import pytest

from test_oracle_pins import _kuhn_interp, kuhn_simplices_of_cell, qp_simplex_distance, to_xyz_order


def _case(seed, rdims, edims):
    rng = np.random.default_rng([41, seed])
    ref = rng.uniform(0.9, 2.0, size=rdims[::-1])            # arrays are [z, y, x]
    ev = rng.uniform(0.9, 2.0, size=edims[::-1])
    return ref, ev


def test_same_geometry_equals_the_same_grid_oracle(oracle_mod):
    rng = np.random.default_rng(3)
    ref = rng.uniform(0.8, 2.0, size=(5, 6, 7))
    ev = ref * 1.03 + rng.normal(0, 0.06, size=ref.shape)
    dims, sp = (7, 6, 5), (2.0, 2.5, 3.0)
    for mode, cutoff in ((0, 0.0), (1, 0.3), (0, 0.6)):
        a = oracle_mod.gamma(ref, ev, dims, sp, 0.03, 3.0, mode, cutoff)
        for form in ("all", "shell"):
            b = oracle_mod.gamma_general(ref, dims, sp, (5.0, -3.0, 11.0), ev, dims, sp, (5.0, -3.0, 11.0), 0.03, 3.0, mode,
                                         cutoff, form=form)
            assert np.array_equal(np.isnan(a), np.isnan(b))
            m = ~np.isnan(a)
            assert np.abs(a[m] - b[m]).max() <= 1e-13


def test_integer_voxel_origin_shift_is_an_index_shift(oracle_mod):
    """Reference grid = a sub-block of the evaluation grid's lattice (origin shifted by whole voxels): the general
    oracle must return what the same-grid oracle returns for those voxels of the embedding grid."""
    rng = np.random.default_rng(5)
    edims, sp, k, rdims = (9, 8, 7), (2.0, 2.5, 1.5), (2, 1, 3), (5, 6, 3)
    ev = rng.uniform(0.8, 2.0, size=edims[::-1])
    ref = rng.uniform(0.8, 2.0, size=rdims[::-1])
    emb = np.zeros(edims[::-1])
    emb[k[2]:k[2] + rdims[2], k[1]:k[1] + rdims[1], k[0]:k[0] + rdims[0]] = ref
    vox = [(x + k[0]) + edims[0] * ((y + k[1]) + edims[1] * (z + k[2]))
           for z in range(rdims[2]) for y in range(rdims[1]) for x in range(rdims[0])]
    want = oracle_mod.gamma(emb, ev, edims, sp, 0.03, 2.0, 0, 0.0, norm_dose=2.0, voxels=vox)
    origin_e = np.array([-4.0, 7.5, 3.0])
    origin_r = origin_e + np.array(k) * np.array(sp)
    got = oracle_mod.gamma_general(ref, rdims, sp, origin_r, ev, edims, sp, origin_e, 0.03, 2.0, 0, 0.0, norm_dose=2.0)
    assert np.abs(got - want).max() <= 1e-13


def test_ramp_closed_form_unequal_spacings_fractional_offset(oracle_mod):
    """D_e = a + g.x is reproduced exactly by any simplicial interpolant; for a reference point with dose D_r the
    distance to that hyperplane is |D_r - D_e(x_r)| / sqrt(dD^2 + dd^2 |g|^2) (Eq. 1), whatever the
    two grids are, as long as the foot point stays inside the evaluation grid."""
    g = np.array([0.05, -0.02, 0.03])
    a, dD, dta = 10.0, 0.06, 3.0
    edims, esp, eorg = (14, 12, 16), (2.0, 3.5, 1.25), np.array([-13.0, -19.0, -10.0])
    rdims, rsp, rorg = (5, 4, 6), (1.7, 2.3, 0.9), np.array([-3.3, -4.1, -2.2])         # fractional everywhere
    ax = [eorg[i] + np.arange(edims[i]) * esp[i] for i in range(3)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    ev = a + g[0] * X + g[1] * Y + g[2] * Z
    rx = [rorg[i] + np.arange(rdims[i]) * rsp[i] for i in range(3)]
    RZ, RY, RX = np.meshgrid(rx[2], rx[1], rx[0], indexing="ij")
    rng = np.random.default_rng(9)
    c = rng.uniform(-0.1, 0.1, size=RX.shape)
    ref = a + g[0] * RX + g[1] * RY + g[2] * RZ + c
    closed = np.abs(c) / np.sqrt(dD ** 2 + dta ** 2 * (g @ g))
    for form in ("all", "shell"):
        got, clo = oracle_mod.gamma_general(ref, rdims, rsp, rorg, ev, edims, esp, eorg, dD, dta, 0, 0.0, norm_dose=1.0,
                                            form=form, return_closest=True)
        assert np.abs(got.reshape(RX.shape) - closed).max() <= 1e-12
        # the closest point is the foot of the perpendicular: x_r + (D_r - D_e(x_r)) g dd^2 / (dD^2 + dd^2 |g|^2)
        foot = (np.stack([RX, RY, RZ], axis=-1) + (c / (dD ** 2 + dta ** 2 * (g @ g)) * dta ** 2)[..., None] * g).reshape(-1, 3)
        assert np.abs(clo[:, :3] - foot).max() <= 1e-9
        assert np.abs(clo[:, 3] - (a + foot @ g)).max() <= 1e-9


@pytest.mark.parametrize("seed,rdims,rsp,rorg,edims,esp,eorg,dd,dta", [
    (1, (3, 2, 2), (1.7, 2.1, 1.3), (0.4, 0.9, 0.2), (3, 3, 3), (2.0, 2.5, 3.0), (0.0, 0.0, 0.0), 0.03, 3.0),
    (2, (2, 3, 2), (3.1, 1.1, 2.7), (-2.5, 1.2, -1.0), (4, 3, 3), (1.5, 2.0, 2.5), (0.0, 0.0, 0.0), 0.05, 2.0),   # points outside the grid too
    (3, (2, 2, 2), (5.0, 5.0, 5.0), (0.5, 0.5, 0.5), (3, 4, 2), (3.0, 2.0, 4.0), (0.0, 0.0, 0.0), 0.02, 1.5),
])
def test_bruteforce_all_simplices_library_qp(oracle_mod, seed, rdims, rsp, rorg, edims, esp, eorg, dd, dta):
    """gamma[v] == min over ALL Kuhn simplices of the evaluation grid of a library-QP distance (no radius, no
    pruning), the reference point being anywhere relative to the evaluation lattice; and the closest point is ON
    the surface (independent Kuhn interpolator) at normalised distance gamma."""
    ref, ev = _case(seed, rdims, edims)
    ev_xyz = to_xyz_order(ev)
    dnorm = ref.max()
    dD = dd * dnorm
    for form in ("all", "shell"):
        got, clo = oracle_mod.gamma_general(ref, rdims, rsp, rorg, ev, edims, esp, eorg, dd, dta, 0, 0.0, form=form,
                                            return_closest=True)
        got = got.reshape(ref.shape)
        clo = clo.reshape(ref.shape + (4,))
        for vz, vy, vx in itertools.product(*[range(n) for n in ref.shape]):
            xr = np.array(rorg) + np.array([vx, vy, vz]) * np.array(rsp)
            Dr = ref[vz, vy, vx]
            best = np.inf
            for c in itertools.product(*[range(n - 1) for n in edims]):
                for chain in kuhn_simplices_of_cell(c, 3):
                    pts = np.zeros((4, 4))
                    for i, uu in enumerate(chain):
                        pts[i, :3] = (np.array(eorg) + uu * np.array(esp) - xr) / dta
                        pts[i, 3] = (ev_xyz[tuple(uu)] - Dr) / dD
                    best = min(best, qp_simplex_distance(pts))
            assert got[vz, vy, vx] == pytest.approx(best, abs=5e-7)
            p = clo[vz, vy, vx]
            idx = (p[:3] - np.array(eorg)) / np.array(esp)
            assert np.all(idx >= -1e-12) and np.all(idx <= np.array(edims) - 1 + 1e-12)
            assert _kuhn_interp(ev_xyz, [np.clip(idx, 0, np.array(edims) - 1)])[0] == pytest.approx(p[3], abs=1e-10)
            dist = np.sqrt(((p[:3] - xr) ** 2).sum() / dta ** 2 + ((p[3] - Dr) / dD) ** 2)
            assert dist == pytest.approx(got[vz, vy, vx], abs=1e-12)


def test_shell_form_equals_every_cell_form_on_a_resampled_case(oracle_mod):
    """The pruned form (what the large comparisons use) against the unpruned definition on a case with deep searches:
    evaluation on a finer, shifted grid, rough doses."""
    rng = np.random.default_rng(17)
    rdims, rsp, rorg = (6, 5, 4), (3.0, 3.0, 3.0), (1.0, 2.0, 0.5)
    edims, esp, eorg = (11, 10, 8), (2.0, 2.0, 2.0), (-0.7, 0.3, -1.1)
    ref = rng.uniform(0.5, 2.0, size=rdims[::-1])
    ev = rng.uniform(0.5, 2.0, size=edims[::-1])
    for mode, cutoff in ((0, 0.0), (1, 0.4)):
        a = oracle_mod.gamma_general(ref, rdims, rsp, rorg, ev, edims, esp, eorg, 0.02, 2.0, mode, cutoff, form="all")
        b, clo = oracle_mod.gamma_general(ref, rdims, rsp, rorg, ev, edims, esp, eorg, 0.02, 2.0, mode, cutoff, form="shell",
                                          return_closest=True)
        assert np.array_equal(np.isnan(a), np.isnan(b))
        m = ~np.isnan(a)
        assert np.array_equal(a[m], b[m])
        assert np.nanmax(a) > 1.5                               # the search really leaves the first shell
        assert np.array_equal(np.isnan(clo[:, 0]), np.isnan(a))


def test_general_oracle_rejects_invalid_arguments(oracle_mod):
    a = np.ones((2, 2, 2))
    g = ((2, 2, 2), (1, 1, 1), (0, 0, 0))
    with pytest.raises(ValueError):
        oracle_mod.gamma_general(a, *g, a, *g, -0.03, 3.0)
    with pytest.raises(ValueError):
        oracle_mod.gamma_general(a, *g, np.ones((2, 2)), (2, 2, 1), (1, 1, 1), (0, 0, 0), 0.03, 3.0)   # eval axis of size 1
    with pytest.raises(ValueError):
        oracle_mod.gamma_general(a, *g, a, *g, 0.03, 3.0, form="nope" if False else "all", cutoff=1.5)
