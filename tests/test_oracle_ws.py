"""Pins of the oracle's Wigner-Seitz defect count (ref. [34]): constructed
defects, the closed form of the bcc Wigner-Seitz cell, and an independent nearest-site search (scipy)."""
import numpy as np
import pytest
from scipy.spatial import cKDTree

import oracle
from paper_2305_08140_b200 import workloads as wl


def test_thermal_lattice_has_no_defects():
    site, pos, box, pbc, _ = wl.defective_lattice(5, seed=1, n_vacancies=0, n_interstitials=0)
    nearest, occ, (nv, ni) = oracle.wigner_seitz(site, pos, box, pbc)
    assert np.array_equal(nearest, np.arange(site.shape[1])) and np.all(occ == 1) and (nv, ni) == (0, 0)


def test_constructed_defects_are_found():
    site, pos, box, pbc, info = wl.defective_lattice(6, seed=2, n_vacancies=5, n_interstitials=3, n_frenkel=4)
    nearest, occ, (nv, ni) = oracle.wigner_seitz(site, pos, box, pbc)
    assert (nv, ni) == (9, 7)
    assert sorted(np.flatnonzero(occ == 0)) == info["vacant"]
    assert sorted(np.flatnonzero(occ == 2)) == info["double"]
    assert occ.sum() == pos.shape[1] and occ.max() == 2


def test_periodic_wrap_and_open_axis():
    a = wl.A0_CONFIG
    site = wl.bcc_lattice(4, 4, 4)
    box = np.diag([4 * a] * 3).ravel()
    pos = site.copy()
    pos[0, 0] = 4 * a - 0.3          # site 0 sits at the origin: 0.3 A across the periodic face
    n1, _, c1 = oracle.wigner_seitz(site, pos, box, [1, 1, 1])
    assert n1[0] == 0 and c1 == (0, 0)
    n2, occ2, c2 = oracle.wigner_seitz(site, pos, box, [0, 1, 1])  # open in x: nearest site is at x = 3.5 a
    assert n2[0] != 0 and site[0, n2[0]] == 3.5 * a and c2 == (1, 1)


def test_bcc_wigner_seitz_cell_closed_form():
    # the W-S cell of a bcc site is the truncated octahedron |x|,|y|,|z| <= a/2, |x|+|y|+|z| <= 3a/4
    a = wl.A0_CONFIG
    site = wl.bcc_lattice(4, 4, 4)
    box = np.diag([4 * a] * 3).ravel()
    g = wl.rng(11, 9)
    p = g.uniform(-0.75 * a, 0.75 * a, size=(3, 4000))
    c = site[:, [2 * (1 * 16 + 1 * 4 + 1)]]  # corner site of cell (1,1,1)
    inside = (np.abs(p).max(axis=0) < 0.5 * a) & (np.abs(p).sum(axis=0) < 0.75 * a)
    margin = np.minimum(0.5 * a - np.abs(p).max(axis=0), 0.75 * a - np.abs(p).sum(axis=0))
    ok = np.abs(margin) > 1e-9
    nearest, _, _ = oracle.wigner_seitz(site, c + p, box, [1, 1, 1])
    assert inside.mean() == pytest.approx(0.5 / 1.5 ** 3, rel=0.15)  # cell volume a^3/2 of the (1.5 a)^3 sampling cube
    assert np.array_equal((nearest == 2 * 21)[ok], inside[ok])


def test_against_kdtree():
    site, pos, box, pbc, _ = wl.defective_lattice((5, 6, 7), seed=3, n_vacancies=10, n_interstitials=10,
                                                  n_frenkel=10, sigma=0.5)
    L = box[[0, 4, 8]]
    _, idx = cKDTree(np.mod(site.T, L), boxsize=L).query(np.mod(pos.T, L))
    nearest, occ, _ = oracle.wigner_seitz(site, pos, box, pbc)
    assert np.array_equal(nearest, idx)
    assert np.array_equal(occ, np.bincount(idx, minlength=site.shape[1]))
    sel = np.arange(0, pos.shape[1], 7, dtype=np.int32)
    n2, _, _ = oracle.wigner_seitz(site, pos, box, pbc, sel=sel)
    assert np.array_equal(n2[sel], nearest[sel]) and np.all(np.delete(n2, sel) == -1)
