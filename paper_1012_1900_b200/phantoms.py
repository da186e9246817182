"""Seeded synthetic dose grids for the five BASELINE.json configs.

This module holds NO gamma-index arithmetic: it only manufactures the input
dose grids (reference, evaluation) and names the comparison criteria.  Both the
CUDA path and the CPU oracle are fed from here (tests and bench.py pass the
arrays to each side); neither side imports the other.

The grids stand in for the paper's eight IMRT patient dose pairs (Monte-Carlo
reference vs pencil-beam evaluation, section 3.1), which are not
available.  The recipe follows SURVEY.md section 8(d) and BASELINE.json
``configs``; it is restated in DESIGN.md ("Input recipe").

Conventions
-----------
* arrays are C-contiguous with shape (nz, ny, nx): x is the fastest axis, i.e.
  ``lin = ix + nx*(iy + ny*iz)``;
* voxel centres sit at ``x_a = (i_a - (n_a-1)/2) * h_a`` (mm);
* everything is computed in float64 and cast to float32 at the end;
* RNG: ``numpy.random.default_rng([seed, config_id, stream_id])``.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
from scipy.ndimage import map_coordinates
from scipy.special import erf, ndtr

__all__ = ["Case", "GeneralCase", "make_case", "make_general_case", "CASE_NAMES", "resample_shifted", "beam_phantom",
           "blob_phantom_2d"]


@dataclass
class Case:
    """One gamma-index problem: two dose grids on the same grid plus criteria."""

    name: str
    ref: np.ndarray                 # float32, shape (nz, ny, nx)
    eval: np.ndarray                # float32, same shape
    dims: tuple                     # (nx, ny, nz)
    spacing_mm: tuple               # (dx, dy, dz)
    dd: float                       # dose-difference criterion, fraction
    dta_mm: float                   # distance-to-agreement criterion, mm
    mode: int = 0                   # 0 global, 1 local
    cutoff: float = 0.10            # low-dose cutoff, fraction of max(ref)
    meta: dict = field(default_factory=dict)


def _axes(dims, spacing):
    nx, ny, nz = dims
    dx, dy, dz = spacing
    x = (np.arange(nx, dtype=np.float64) - (nx - 1) / 2.0) * dx
    y = (np.arange(ny, dtype=np.float64) - (ny - 1) / 2.0) * dy
    z = (np.arange(nz, dtype=np.float64) - (nz - 1) / 2.0) * dz
    return x, y, z


def _edge_profile(s, half_width, sigma):
    """Flat field of half-width `half_width` (mm) with erf penumbra `sigma`."""
    k = 1.0 / (np.sqrt(2.0) * sigma)
    return 0.5 * (erf((half_width - s) * k) + erf((half_width + s) * k))


# --------------------------------------------------------------------------
# config 1: 2D blobs + plateau
# --------------------------------------------------------------------------
def blob_phantom_2d(dims, spacing, seed=0, config_id=1):
    nx, ny, nz = dims
    assert nz == 1
    x, y, _ = _axes(dims, spacing)
    X, Y = np.meshgrid(x, y, indexing="xy")      # shape (ny, nx)
    rng = np.random.default_rng([seed, config_id, 0])
    half_x = (nx - 1) / 2.0 * spacing[0]
    half_y = (ny - 1) / 2.0 * spacing[1]
    d = np.zeros_like(X)
    for _ in range(4):
        cx = rng.uniform(-0.6, 0.6) * half_x
        cy = rng.uniform(-0.6, 0.6) * half_y
        sx = rng.uniform(5.0, 20.0)
        sy = rng.uniform(5.0, 20.0)
        amp = rng.uniform(0.5, 1.0)
        d += amp * np.exp(-0.5 * (((X - cx) / sx) ** 2 + ((Y - cy) / sy) ** 2))
    # axis-aligned rectangular plateau, half-widths 25 x 15 mm, erf edges sigma 3 mm
    px = rng.uniform(-0.2, 0.2) * half_x
    py = rng.uniform(-0.2, 0.2) * half_y
    d += 0.8 * _edge_profile(X - px, 25.0, 3.0) * _edge_profile(Y - py, 15.0, 3.0)
    d *= 2.0 / d.max()
    return d.reshape(1, ny, nx)


# --------------------------------------------------------------------------
# configs 2-5: seven coplanar modulated beams in an elliptical body
# --------------------------------------------------------------------------
def _bixel_masses(c, nb, bixel_mm, sigma):
    """Mass of N(c, sigma) in each of the nb bixels along one axis: shape (nb,) + c.shape."""
    edges = (np.arange(nb + 1) - nb / 2.0) * bixel_mm
    cdf = ndtr((edges.reshape((-1,) + (1,) * c.ndim) - c[None]) / sigma)
    return cdf[1:] - cdf[:-1]


def beam_phantom(dims, spacing, seed=0, config_id=2):
    """7 coplanar beams, 60x60 mm fields, erf penumbra, exponential attenuation."""
    nx, ny, nz = dims
    x, y, z = _axes(dims, spacing)
    X, Y = np.meshgrid(x, y, indexing="xy")      # (ny, nx): one axial slice
    rng = np.random.default_rng([seed, 2, 0])    # same fluence maps for configs 2-5
    a_body, b_body = 150.0, 100.0                # ellipse x^2/150^2 + y^2/100^2 = 1
    inside_body = (X / a_body) ** 2 + (Y / b_body) ** 2 <= 1.0
    sigma_pen, half_field, mu = 3.0, 30.0, 0.005
    dose = np.zeros((nz, ny, nx), dtype=np.float64)
    zprof_cache = _edge_profile(z, half_field, sigma_pen)    # (nz,)
    for b in range(7):
        th = 2.0 * np.pi * b / 7.0
        # beam travels along direction (cos th, sin th); source side is -direction
        dirx, diry = np.cos(th), np.sin(th)
        s_lat = -X * diry + Y * dirx             # lateral in-plane coordinate
        along = X * dirx + Y * diry              # coordinate along the beam
        # entry point of the ray on the ellipse: solve for lambda < 0 side
        # point(l) = p + l*dir, on ellipse: A l^2 + B l + C = 0
        A = (dirx / a_body) ** 2 + (diry / b_body) ** 2
        # ray through (X,Y): base point is the foot with along = 0
        bx = -s_lat * diry
        by = s_lat * dirx
        B = 2.0 * (bx * dirx / a_body ** 2 + by * diry / b_body ** 2)
        C = (bx / a_body) ** 2 + (by / b_body) ** 2 - 1.0
        disc = np.maximum(B * B - 4.0 * A * C, 0.0)
        l_entry = (-B - np.sqrt(disc)) / (2.0 * A)
        depth = np.maximum(along - l_entry, 0.0)
        weights = rng.uniform(0.5, 1.5, size=(8, 8))
        lat_prof = _edge_profile(s_lat, half_field, sigma_pen)
        atten = np.exp(-mu * depth)
        base2d = np.where(inside_body, lat_prof * atten, 0.0)          # (ny, nx)
        # fluence = 8x8 bixel map (7.5 mm bixels) convolved analytically with a Gaussian
        # (sigma 10 mm): sum_ij W_ij P_i(s_lat) P_j(z), and 1.0 outside the 8x8 field so
        # that the modulation is a continuous function.  Separable in (s_lat, z).
        pu = _bixel_masses(s_lat, 8, 7.5, 10.0)                # (8, ny, nx)
        pt = _bixel_masses(z, 8, 7.5, 10.0)                    # (8, nz)
        au = np.einsum("ij,iyx->jyx", weights, pu)             # (8, ny, nx)
        mass_u = pu.sum(axis=0)                                # (ny, nx)
        mass_t = pt.sum(axis=0)                                # (nz,)
        for iz in range(nz):
            flu = np.tensordot(pt[:, iz], au, axes=(0, 0)) + (1.0 - mass_u * mass_t[iz])
            dose[iz] += base2d * zprof_cache[iz] * flu
    dose *= 2.0 / dose.max()
    return dose


def resample_shifted(ref64, spacing, shift_mm):
    """(Multi)linear resample of the discretised ref at x - shift, edge-clamped."""
    nz, ny, nx = ref64.shape
    dx, dy, dz = spacing
    sx, sy, sz = shift_mm
    iz, iy, ix = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                             np.arange(nx, dtype=np.float64), indexing="ij")
    coords = [iz - (sz / dz if nz > 1 else 0.0), iy - sy / dy, ix - sx / dx]
    return map_coordinates(ref64, coords, order=1, mode="nearest")


def _perturb(ref64, spacing, shift_mm, scale, noise_frac, rng):
    ev = scale * resample_shifted(ref64, spacing, shift_mm)
    ev = ev + rng.normal(0.0, noise_frac * ref64.max(), size=ref64.shape)
    return ev


@dataclass
class GeneralCase:
    """A gamma-index problem whose evaluation dose lives on its own grid."""

    name: str
    ref: np.ndarray
    ref_dims: tuple
    ref_spacing_mm: tuple
    ref_origin_mm: tuple            # position of the centre of reference voxel (0, 0, 0)
    eval: np.ndarray
    eval_dims: tuple
    eval_spacing_mm: tuple
    eval_origin_mm: tuple
    dd: float
    dta_mm: float
    mode: int = 0
    cutoff: float = 0.10


def make_general_case(name: str, seed: int = 0) -> GeneralCase:
    """"cfg3_general": the cfg3 reference (128x128x64 at 2.5 mm) against the same beam phantom computed analytically on
    a 2 mm grid (160x160x80) whose origin is displaced by a fraction of a voxel, with cfg3's perturbation (shift, scale,
    noise) and criteria.  "general_small": the same construction on grids the oracle finishes in a second."""
    if name == "cfg3_general":
        rd, rs, ed, es, off = (128, 128, 64), (2.5, 2.5, 2.5), (160, 160, 80), (2.0, 2.0, 2.0), (0.37, -0.81, 0.55)
    elif name == "general_small":
        rd, rs, ed, es, off = (40, 36, 20), (7.5, 7.0, 8.0), (50, 42, 27), (6.0, 6.0, 6.0), (1.3, -2.2, 0.9)
    else:
        raise KeyError(name)
    ref = beam_phantom(rd, rs, seed, 3)
    ev0 = beam_phantom(ed, es, seed, 3)
    ev0 *= 1.0                                   # same analytic phantom: both normalised to 2.0 Gy at their own maximum
    rng = np.random.default_rng([seed, 13, 1])
    ev = _perturb(ev0, es, (2.0, 1.5, -1.0), 0.97, 0.02, rng)
    ro = tuple(-(n - 1) / 2.0 * h for n, h in zip(rd, rs))
    eo = tuple(-(n - 1) / 2.0 * h + o for n, h, o in zip(ed, es, off))
    return GeneralCase(name, ref.astype(np.float32), rd, rs, ro, ev.astype(np.float32), ed, es, eo, 0.02, 2.0, 0, 0.10)


CASE_NAMES = ("cfg1", "cfg2", "cfg3", "cfg4_fine", "cfg4_coarse", "cfg5", "cfg2_small")


def make_case(name: str, seed: int = 0) -> Case:
    """Build one of the named cases (see CASE_NAMES)."""
    if name == "cfg1":
        dims, sp = (64, 64, 1), (2.5, 2.5, 2.5)
        ref = blob_phantom_2d(dims, sp, seed, 1)
        rng = np.random.default_rng([seed, 1, 1])
        ev = _perturb(ref, sp, (0.8, -0.5, 0.0), 1.02, 0.005, rng)
        return Case(name, ref.astype(np.float32), ev.astype(np.float32), dims, sp, 0.03, 3.0, 0, 0.10,
                    {"desc": "2D 64x64, 3%/3mm"})
    if name in ("cfg2", "cfg3", "cfg2_small"):
        dims = (128, 128, 64) if name != "cfg2_small" else (48, 40, 24)
        sp = (2.5, 2.5, 2.5) if name != "cfg2_small" else (7.0, 6.5, 7.5)
        ref = beam_phantom(dims, sp, seed, 2)
        if name == "cfg3":
            rng = np.random.default_rng([seed, 3, 1])
            ev = _perturb(ref, sp, (2.0, 1.5, -1.0), 0.97, 0.02, rng)
            dd, dta = 0.02, 2.0
        else:
            rng = np.random.default_rng([seed, 2, 1])
            ev = _perturb(ref, sp, (1.0, -0.7, 0.5), 1.02, 0.01, rng)
            dd, dta = 0.03, 3.0
        return Case(name, ref.astype(np.float32), ev.astype(np.float32), dims, sp, dd, dta, 0, 0.10,
                    {"desc": "3D beam phantom"})
    if name in ("cfg4_fine", "cfg4_coarse"):
        dims, sp = ((256, 256, 128), (1.25,) * 3) if name == "cfg4_fine" else ((64, 64, 32), (5.0,) * 3)
        ref = beam_phantom(dims, sp, seed, 4)
        rng = np.random.default_rng([seed, 4, 1 if name == "cfg4_fine" else 2])
        ev = _perturb(ref, sp, (1.0, -0.7, 0.5), 1.02, 0.01, rng)
        return Case(name, ref.astype(np.float32), ev.astype(np.float32), dims, sp, 0.03, 3.0, 0, 0.10,
                    {"desc": "resolution sweep"})
    if name == "cfg5":
        dims, sp = (192, 192, 96), (2.0, 2.0, 2.0)
        ref = beam_phantom(dims, sp, seed, 5)
        rng = np.random.default_rng([seed, 5, 1])
        shifted = resample_shifted(ref, sp, (4.0, 0.0, 0.0))
        nz, ny, nx = ref.shape
        ev = ref.copy()
        ev[: nz // 2, : ny // 2, : nx // 2] = shifted[: nz // 2, : ny // 2, : nx // 2]
        ev = 1.05 * ev + rng.normal(0.0, 0.03 * ref.max(), size=ref.shape)
        return Case(name, ref.astype(np.float32), ev.astype(np.float32), dims, sp, 0.01, 1.0, 0, 0.05,
                    {"desc": "load-imbalance stress"})
    raise KeyError(f"unknown case {name!r}; choose from {CASE_NAMES}")
