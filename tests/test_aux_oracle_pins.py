"""Pins for oracle/aux_oracle.py (stats, pair sort, offset table): hand-counted inputs, the table sizes
listed in SURVEY.md section 8(a) (counted there over the full offset space, 8 offsets per octant entry in 3D,
4 in 2D), and brute force over offsets o with the cell bound of DESIGN.md reading 4.  No GPU needed."""
import itertools

import numpy as np
import pytest

from oracle import aux_oracle


def test_stats_hand_counted():
    g = np.array([0.0, 0.5, 1.0, 1.0000001, 2.0, np.nan, 3.999, 4.0, 9.0, np.nan], dtype=np.float32)
    hist, s = aux_oracle.stats(g, 4, 4.0)
    assert s["n_eval"] == 8 and s["n_nan"] == 2
    assert s["n_pass"] == 3                       # 0, 0.5, 1.0 ; 1.0000001 rounds to 1.0000001192 > 1
    assert hist.tolist() == [2, 2, 1, 3]          # [0,1): 0, .5 | [1,2): 1, 1.0000001 | [2,3): 2 | rest
    assert s["max_gamma"] == 9.0
    assert s["sum_gamma"] == pytest.approx(sum(float(x) for x in g[~np.isnan(g)]), rel=1e-15)
    assert s["sum_gamma3"] == pytest.approx(sum(float(x) ** 3 for x in g[~np.isnan(g)]), rel=1e-15)


def test_stats_empty_and_all_nan():
    hist, s = aux_oracle.stats(np.full(5, np.nan, dtype=np.float32), 8, 2.0)
    assert hist.sum() == 0 and s["n_eval"] == 0 and s["n_nan"] == 5 and s["max_gamma"] == 0.0


def test_sort_pairs_is_stable_and_partial_bits():
    k = np.array([0x0201, 0x0102, 0x0101, 0x0202, 0x0101], dtype=np.uint32)
    v = np.arange(5, dtype=np.uint32)
    ks, vs = aux_oracle.sort_pairs(k, v, 0, 32)
    assert ks.tolist() == [0x0101, 0x0101, 0x0102, 0x0201, 0x0202] and vs.tolist() == [2, 4, 1, 0, 3]
    ks, vs = aux_oracle.sort_pairs(k, v, 8, 16)    # by the second byte only, ties keep input order
    assert vs.tolist() == [1, 2, 4, 0, 3]
    f = np.array([3.5, 0.0, 1e-30, 2.25, 7e8], dtype=np.float32)   # non-negative floats order as their bits
    ks, vs = aux_oracle.sort_pairs(f.view(np.uint32), v, 0, 32)
    assert np.array_equal(ks.view(np.float32), np.sort(f))


@pytest.mark.parametrize("dims,sp,dta,sizes", [
    ((128, 128, 64), (2.5, 2.5, 2.5), 3.0, {1: 32, 2: 136, 3: 312, 5: 1256, 10: 8504}),
    ((128, 128, 64), (2.5, 2.5, 2.5), 2.0, {1: 8, 2: 56, 3: 136, 5: 408, 10: 2728}),
    ((192, 192, 96), (2.0, 2.0, 2.0), 1.0, {2: 8, 3: 56, 5: 160, 10: 720}),
    ((64, 64, 1), (2.5, 2.5, 2.5), 3.0, {1: 12, 3: 52, 10: 484}),
])
def test_offset_table_sizes_listed_in_survey(dims, sp, dta, sizes):
    nact = sum(d > 1 for d in dims)
    for R, full_count in sizes.items():
        tab = aux_oracle.offset_table(dims, sp, dta, float(R))
        assert len(tab) * 2 ** nact == full_count
        L2 = [t[0] for t in tab]
        assert L2 == sorted(L2) and tab[0][1:] == (0, 0, 0)


def test_offset_table_equals_bruteforce_over_offsets():
    dims, sp, dta, R = (9, 7, 5), (2.0, 3.0, 2.5), 3.0, 2.2
    h = [s / dta for s in sp]
    cells = set()
    for o in itertools.product(range(-6, 6), repeat=3):
        m = [max(oa, -oa - 1) for oa in o]
        if any(ma > da - 1 for ma, da in zip(m, dims)):
            continue
        if np.sqrt(sum((ma * ha) ** 2 for ma, ha in zip(m, h))) < R:
            cells.add(tuple(m))
    tab = aux_oracle.offset_table(dims, sp, dta, R)
    assert {t[1:] for t in tab} == cells and len(tab) == len(cells)
