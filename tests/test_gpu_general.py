"""Parity of gamma_eval_general (evaluation dose on its own grid, closest point) with the CPU
oracle oracle/gamma_general_oracle.c, through the C-ABI.  Needs a B200: every test is marked `gpu`.
Bar as in test_gpu_parity.py: |dgamma| <= 1e-4 absolute per voxel, identical NaN masks, pass/fail equal outside 1e-4 of 1.
"""
import numpy as np
import pytest
import torch

from paper_1012_1900_b200 import binding, phantoms
from paper_1012_1900_b200.binding import GammaOpts
from test_gpu_parity import assert_parity, assert_parity_local_tiny_doses, f32
from test_oracle_pins import _kuhn_interp, to_xyz_order

pytestmark = pytest.mark.gpu


def f3(v):
    return [f32(x) for x in v]


def gpu_general(ref, rd, rs, ro, ev, ed, es, eo, dd, dta, mode=0, cutoff=0.1, opts=None, closest=True):
    r = torch.from_numpy(np.ascontiguousarray(ref, dtype=np.float32).ravel()).cuda()
    e = torch.from_numpy(np.ascontiguousarray(ev, dtype=np.float32).ravel()).cuda()
    out = binding.gamma_eval_general(r, rd, rs, ro, e, ed, es, eo, dd, dta, mode, cutoff, opts, want_closest=closest)
    torch.cuda.synchronize()
    if closest:
        return out[0].cpu().numpy().astype(np.float64), out[1].cpu().numpy().astype(np.float64)
    return out.cpu().numpy().astype(np.float64)


def cpu_general(oracle_mod, ref, rd, rs, ro, ev, ed, es, eo, dd, dta, mode=0, cutoff=0.1, norm_dose=0.0):
    return oracle_mod.gamma_general(np.asarray(ref, dtype=np.float32), rd, f3(rs), f3(ro), np.asarray(ev, dtype=np.float32), ed,
                                    f3(es), f3(eo), f32(dd), f32(dta), mode, f32(cutoff), f32(norm_dose), return_closest=True)


def check_closest(g, clo, want_g, want_clo, ref, rd, rs, ro, ev, ed, es, eo, dd, dta, mode, what, sample=400):
    """The closest point: NaN exactly where gamma is; at normalised distance gamma from the reference point; on the
    evaluation surface (independent Kuhn interpolator, on a sample); equal to the oracle's wherever that is unique."""
    m = ~np.isnan(want_g)
    assert np.array_equal(np.isnan(clo[:, 0]), ~m), what
    rd = np.array(rd)
    idx = np.flatnonzero(m)
    v = np.stack([idx % rd[0], (idx // rd[0]) % rd[1], idx // (rd[0] * rd[1])], axis=1)
    xr = np.array(f3(ro)) + v * np.array(f3(rs))
    Dr = np.asarray(ref, dtype=np.float32).ravel().astype(np.float64)[idx]
    dnorm = float(np.asarray(ref, dtype=np.float32).max())
    dD = f32(dd) * (dnorm if mode == 0 else Dr)
    dist = np.sqrt((((clo[idx, :3] - xr) / f32(dta)) ** 2).sum(axis=1) + ((clo[idx, 3] - Dr) / dD) ** 2)
    assert np.abs(dist - g[idx]).max() <= 2e-4, f"{what}: closest point is not at distance gamma"
    rng = np.random.default_rng(5)
    ev_xyz = to_xyz_order(np.asarray(ev, dtype=np.float32).astype(np.float64).reshape(ed[2], ed[1], ed[0]))
    pick = rng.choice(idx.size, size=min(sample, idx.size), replace=False)
    fi = (clo[idx[pick], :3] - np.array(f3(eo))) / np.array(f3(es))
    assert np.all(fi >= -1e-3) and np.all(fi <= np.array(ed) - 1 + 1e-3), f"{what}: closest point outside the evaluation grid"
    surf = _kuhn_interp(ev_xyz, np.clip(fi, 0, np.array(ed) - 1))
    tol = 3e-4 * np.max(dD) + 1e-4 * np.abs(surf).max()                         # fp32 coordinates: a few 1e-4 dD
    assert np.abs(surf - clo[idx[pick], 3]).max() <= tol, f"{what}: closest point is not on the surface"
    same = np.linalg.norm(clo[idx] - want_clo[idx], axis=1) <= 1e-2
    assert same.mean() >= 0.97, f"{what}: closest point differs from the oracle's on {100 * (1 - same.mean()):.1f} % of the voxels"


def test_identical_geometry_equals_same_grid_path_and_oracle(oracle_mod):
    c = phantoms.make_case("cfg2_small")
    org = (-11.0, 4.5, 30.0)
    g, clo = gpu_general(c.ref, c.dims, c.spacing_mm, org, c.eval, c.dims, c.spacing_mm, org, c.dd, c.dta_mm, 0, c.cutoff)
    want = oracle_mod.gamma(c.ref, c.eval, c.dims, f3(c.spacing_mm), f32(c.dd), f32(c.dta_mm), 0, f32(c.cutoff))
    assert_parity(g, want, "general path, identical geometry, vs the same-grid oracle")
    r = torch.from_numpy(c.ref.ravel().copy()).cuda()
    e = torch.from_numpy(c.eval.ravel().copy()).cuda()
    base = binding.gamma_eval(r, e, c.dims, c.spacing_mm, c.dd, c.dta_mm, 0, c.cutoff).cpu().numpy().astype(np.float64)
    m = ~np.isnan(want)
    assert np.abs(g[m] - base[m]).max() <= 5e-6
    wg, wc = cpu_general(oracle_mod, c.ref, c.dims, c.spacing_mm, org, c.eval, c.dims, c.spacing_mm, org, c.dd, c.dta_mm, 0, c.cutoff)
    check_closest(g, clo, wg, wc, c.ref, c.dims, c.spacing_mm, org, c.eval, c.dims, c.spacing_mm, org, c.dd, c.dta_mm, 0, "identical")


@pytest.mark.parametrize("name", ["general_small", "cfg3_general"])
def test_resampled_evaluation_grid_full_map_parity(oracle_mod, name):
    """The cfg3 reference against the evaluation dose on a 2 mm grid with a fractional origin offset (and the small
    version of it): every voxel against the oracle, closest points included."""
    c = phantoms.make_general_case(name)
    a = (c.ref, c.ref_dims, c.ref_spacing_mm, c.ref_origin_mm, c.eval, c.eval_dims, c.eval_spacing_mm, c.eval_origin_mm, c.dd,
         c.dta_mm, c.mode, c.cutoff)
    want, wclo = cpu_general(oracle_mod, *a)
    for opts in (None, GammaOpts(table_cap=8)):
        g, clo = gpu_general(*a, opts=opts)
        err = assert_parity(g, want, f"{name} {opts}")
        check_closest(g, clo, want, wclo, *a[:-1], f"{name} {opts}")
    print(f"{name}: max|dgamma| {err:.2e} over {int((~np.isnan(want)).sum())} evaluated voxels, max gamma {np.nanmax(want):.3f}")


@pytest.mark.parametrize("rd,rs,ro,ed,es,eo,dd,dta,mode,cutoff,seed", [
    ((17, 13, 9), (2.0, 3.0, 2.5), (1.1, -0.4, 0.7), (23, 19, 12), (1.5, 2.0, 2.5), (0.0, 0.0, 0.0), 0.03, 3.0, 0, 0.1, 1),
    ((17, 13, 9), (2.0, 3.0, 2.5), (1.1, -0.4, 0.7), (23, 19, 12), (1.5, 2.0, 2.5), (0.0, 0.0, 0.0), 0.02, 4.0, 1, 0.0, 2),   # local
    ((9, 8, 7), (4.0, 4.0, 4.0), (-6.0, -5.0, -9.0), (12, 10, 11), (2.0, 2.5, 1.5), (0.0, 0.0, 0.0), 0.03, 2.0, 0, 0.0, 3),   # points outside the grid
    ((1, 1, 5), (1.0, 1.0, 3.3), (7.2, 6.1, 0.4), (9, 8, 10), (2.0, 2.0, 2.0), (0.0, 0.0, 0.0), 0.03, 3.0, 0, 0.0, 4),        # a line of reference points
    ((6, 5, 4), (3.0, 3.0, 3.0), (0.0, 0.0, 0.0), (2, 2, 2), (20.0, 15.0, 10.0), (0.0, 0.0, 0.0), 0.05, 5.0, 0, 0.0, 5),      # one evaluation cell
    ((11, 7, 5), (0.9, 0.9, 0.9), (3.3, 3.3, 3.3), (30, 6, 4), (0.5, 4.0, 4.0), (0.0, 0.0, 0.0), 0.03, 2.5, 0, 0.2, 6),       # strongly anisotropic
])
@pytest.mark.parametrize("opts", [None, GammaOpts(table_cap=3), GammaOpts(table_cap=4096)])
def test_random_geometries(oracle_mod, rd, rs, ro, ed, es, eo, dd, dta, mode, cutoff, seed, opts):
    rng = np.random.default_rng([seed, 29])
    ref = rng.uniform(0.3, 2.0, size=rd[::-1]).astype(np.float32)
    ev = rng.uniform(0.3, 2.0, size=ed[::-1]).astype(np.float32)
    a = (ref, rd, rs, ro, ev, ed, es, eo, dd, dta, mode, cutoff)
    want, wclo = cpu_general(oracle_mod, *a)
    g, clo = gpu_general(*a, opts=opts)
    assert_parity(g, want, f"{rd}->{ed} {opts}")
    check_closest(g, clo, want, wclo, *a[:-1], f"{rd}->{ed} {opts}", sample=200)
    g2 = gpu_general(*a, opts=opts, closest=False)                     # without the second output: same gamma
    assert np.array_equal(g, g2, equal_nan=True)


def test_ramp_closed_form_on_the_device():
    """D_e = a + g.x on one grid, reference points on another: gamma = |D_r - D_e(x_r)| / sqrt(dD^2 + dd^2 |g|^2) and
    the closest point is the foot of the perpendicular (Eq. 1)."""
    grad = np.array([0.05, -0.02, 0.03])
    a0, dD, dta = 10.0, 0.06, 3.0
    ed, es, eo = (40, 36, 44), (2.0, 3.5, 1.25), np.array([-39.0, -61.0, -27.0])
    rd, rs, ro = (9, 8, 10), (1.7, 2.3, 0.9), np.array([-6.3, -7.1, -4.2])
    ax = [f32(eo[i]) + np.arange(ed[i]) * f32(es[i]) for i in range(3)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    ev = (a0 + grad[0] * X + grad[1] * Y + grad[2] * Z).astype(np.float32)
    rx = [f32(ro[i]) + np.arange(rd[i]) * f32(rs[i]) for i in range(3)]
    RZ, RY, RX = np.meshgrid(rx[2], rx[1], rx[0], indexing="ij")
    rng = np.random.default_rng(9)
    c = rng.uniform(-0.1, 0.1, size=RX.shape)
    ref = (a0 + grad[0] * RX + grad[1] * RY + grad[2] * RZ + c).astype(np.float32)
    # the surface is the interpolant of the ROUNDED doses: compare with the closed form to the size of that rounding
    g, clo = gpu_general(ref, rd, rs, ro, ev, ed, es, eo, dD, dta, 0, 0.0, GammaOpts(norm_dose=1.0))
    resid = ref.astype(np.float64) - (a0 + grad[0] * RX + grad[1] * RY + grad[2] * RZ)
    closed = np.abs(resid) / np.sqrt(f32(dD) ** 2 + dta ** 2 * (grad @ grad))
    assert np.abs(g.reshape(RX.shape) - closed).max() <= 3e-4          # fp32 doses near 10 Gy: ulp 1e-6 Gy = 2e-5 dD
    foot = (np.stack([RX, RY, RZ], axis=-1) + (resid / (f32(dD) ** 2 + dta ** 2 * (grad @ grad)) * dta ** 2)[..., None] * grad)
    assert np.abs(clo[:, :3] - foot.reshape(-1, 3)).max() <= 5e-3


def test_general_argument_errors():
    one = torch.ones(8, device="cuda")
    with pytest.raises(binding.GammaError):
        binding.gamma_eval_general(one, (2, 2, 2), (1, 1, 1), (0, 0, 0), one, (2, 2, 2), (1, 1, 1), (0, 0, 0), -0.03, 3.0)
    with pytest.raises(binding.GammaError):                         # an evaluation axis of size 1
        binding.gamma_eval_general(one, (2, 2, 2), (1, 1, 1), (0, 0, 0), one, (4, 2, 1), (1, 1, 1), (0, 0, 0), 0.03, 3.0)
    with pytest.raises(binding.GammaError):
        binding.gamma_eval_general(one, (2, 2, 2), (1, 0, 1), (0, 0, 0), one, (2, 2, 2), (1, 1, 1), (0, 0, 0), 0.03, 3.0)
    with pytest.raises(binding.GammaError):
        binding.gamma_eval_general(one, (2, 2, 2), (1, 1, 1), (0, float("nan"), 0), one, (2, 2, 2), (1, 1, 1), (0, 0, 0), 0.03, 3.0)


@pytest.mark.parametrize("geometry", ["identical", "general_small"])
def test_general_path_local_mode_zero_and_negative_reference_dose(oracle_mod, geometry):
    """SURVEY.md 8(b) / reading 9 on gamma_eval_general: reference doses of zero and below under the local criterion with
    cutoff 0 are NaN (gamma and closest point), everything else meets the oracle."""
    if geometry == "identical":
        c = phantoms.make_case("cfg2_small")
        ref, rd, rs, ro, ev, ed, es, eo, dd, dta = c.ref.copy(), c.dims, c.spacing_mm, (0.0, 0.0, 0.0), c.eval, c.dims, \
            c.spacing_mm, (0.0, 0.0, 0.0), c.dd, c.dta_mm
    else:
        q = phantoms.make_general_case("general_small")
        ref, rd, rs, ro, ev, ed, es, eo, dd, dta = q.ref.copy(), q.ref_dims, q.ref_spacing_mm, q.ref_origin_mm, q.eval, \
            q.eval_dims, q.eval_spacing_mm, q.eval_origin_mm, q.dd, q.dta_mm
    rng = np.random.default_rng(4)
    inside = np.flatnonzero(ref.ravel() > 0.5)
    ref.ravel()[rng.choice(inside, size=9, replace=False)] = np.float32(-0.02)
    assert (ref == 0).sum() > 500
    wg, wc = cpu_general(oracle_mod, ref, rd, rs, ro, ev, ed, es, eo, dd, dta, 1, 0.0)
    assert np.array_equal(np.isnan(wg), ref.ravel() <= 0)
    g, clo = gpu_general(ref, rd, rs, ro, ev, ed, es, eo, dd, dta, 1, 0.0)
    what = f"general path ({geometry}), local mode, zero / negative reference dose"
    assert np.array_equal(np.isnan(clo[:, 0]), np.isnan(wg))
    if geometry == "identical":
        # same grid: the exact-arithmetic helper applies to the voxels whose tiny D_r defeats the float64 oracle (reading 21)
        err, err_exact, n_ill, n_off = assert_parity_local_tiny_doses(g, wg, ref, ev, rd, rs, dd, dta, what, "general-identical")
        print(f"{what}: max|dgamma| {err:.2e}; {n_ill} voxels with tiny D_r ({n_off} where the oracle is off), vs exact {err_exact:.2e}")
    else:
        # own evaluation grid: the oracle where float64 can decide (D_r >= 1e-4 D_norm), the masks and the one-sided bound
        # (the oracle can only over-estimate) everywhere
        assert np.array_equal(np.isnan(g), np.isnan(wg))
        r = ref.ravel().astype(np.float64)
        well = ~np.isnan(wg) & (r >= 1e-4 * r.max())
        assert_parity(np.where(well, g, np.nan), np.where(well, wg, np.nan), what)
        ill = ~np.isnan(wg) & ~well
        assert np.all(g[ill] <= wg[ill] + 1e-4)
