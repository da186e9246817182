#!/usr/bin/env python3
"""Writes tests/golden/work_model.json: per BASELINE.json config, the quantities of the algorithmic work model
of SURVEY.md section 8(d), computed by the CPU oracle ALONE (this script imports only oracle/ and the seeded
input generators; it never touches the CUDA path).

    N          grid voxels
    M          evaluated voxels (reference dose >= cutoff * max)
    sum_Ns     sum over evaluated voxels of N_s(v) = #{in-grid cells o : L_cell(o) < gamma[v]}: the visits an
               exact bound-ordered search cannot skip (work per voxel ~ gamma^n)
    sum_touch  the part of sum_Ns that are cells touching the voxel (L_cell = 0)
    n_pass, sum_gamma, sum_gamma3, max_gamma   oracle results, for cross-checks of gamma_stats

Run from the repo root:  python tests/golden/make_work_model.py [cfg names...]
Large configs (cfg4_fine, cfg5) take minutes on 8 cores.
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1012_1900_b200 import phantoms  # noqa: E402  (input generators only: no gamma arithmetic there)

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "work_model.json")


def touching_cells(dims, lin):
    """number of in-grid cells that contain voxel lin as a corner"""
    nx, ny, nz = dims
    ix, iy, iz = lin % nx, (lin // nx) % ny, lin // (nx * ny)
    cnt = np.ones_like(lin)
    for i, n in ((ix, nx), (iy, ny), (iz, nz)):
        if n > 1:
            cnt = cnt * ((i >= 1).astype(np.int64) + (i <= n - 2).astype(np.int64))
    return cnt


def main():
    names = sys.argv[1:] or ["cfg1", "cfg2", "cfg3", "cfg4_coarse", "cfg4_fine", "cfg5", "cfg2_small"]
    model = json.load(open(OUT)) if os.path.exists(OUT) else {}
    oracle.build()
    for name in names:
        c = phantoms.make_case(name)
        f = lambda x: float(np.float32(x))
        g, vis = oracle.gamma(c.ref, c.eval, c.dims, [f(s) for s in c.spacing_mm], f(c.dd), f(c.dta_mm), c.mode,
                              f(c.cutoff), return_visits=True)
        m = ~np.isnan(g)
        lin = np.flatnonzero(m)
        touch = np.where(g[m] > 0.0, touching_cells(c.dims, lin), 0)
        model[name] = {
            "N": int(g.size), "M": int(m.sum()), "sum_Ns": int(vis[m].sum()), "sum_touch": int(touch.sum()),
            "n_pass": int((g[m] <= 1.0).sum()), "n_within_1e-4_of_1": int((np.abs(g[m] - 1.0) <= 1e-4).sum()),
            "sum_gamma": float(g[m].sum()), "sum_gamma3": float((g[m] ** 3).sum()), "max_gamma": float(g[m].max()),
        }
        print(name, model[name], flush=True)
        json.dump(model, open(OUT, "w"), indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
