"""Pins of the oracle's neighbour search: brute force with explicit images is the
definition; its own cell list is validated against it; bcc shell counts are textbook."""
import os

import numpy as np
import pytest

import oracle
from paper_2305_08140_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _sets(nn, nl):
    return [sorted(nl[i, :nn[i]].tolist()) for i in range(len(nn))]


def test_bcc_shell_counts():
    rows = [l.split() for l in open(os.path.join(GOLD, "bcc_shells.txt")) if not l.startswith("#")]
    a = wl.A0_CONFIG
    w = wl.thermal_bulk(6, seed=1)                # perfect lattice, box 18.99 A
    total = 0
    for k2, mult in rows:
        total += int(mult)
        rc = 0.5 * a * np.sqrt(float(k2)) + 1e-6  # just beyond this shell
        if rc >= 0.5 * w.box[0]:
            break
        nn, _ = oracle.neighbors(w.pos, w.box, w.pbc, rc)
        assert np.all(nn == total), (k2, total)
    # the counts the hot path is sized for (SURVEY 8 header): 58 < 6 A, 14 < 4 A, 26 < 5 A, 88 < 7 A
    for rc, cnt in ((6.0, 58), (4.0, 14), (5.0, 26), (7.0, 88)):
        nn, _ = oracle.neighbors(w.pos, w.box, w.pbc, rc)
        assert np.all(nn == cnt)


def test_strict_inequality_at_the_cutoff():
    pos = np.array([[1.0, 4.0], [1.0, 1.0], [1.0, 1.0]])
    box = np.diag([50.0, 50, 50]).ravel()
    assert oracle.neighbors(pos, box, [0, 0, 0], 3.0)[0].tolist() == [0, 0]          # r == rc excluded
    assert oracle.neighbors(pos, box, [0, 0, 0], 3.0 + 1e-12)[0].tolist() == [1, 1]


def test_cell_list_equals_brute_force_on_config1():
    w = wl.config1()
    for rc in (4.0, 6.0, 7.0):
        nb, lb, db = oracle.neighbors(w.pos, w.box, w.pbc, rc, use_cell=False, want_d=True)
        nc, lc, dc = oracle.neighbors(w.pos, w.box, w.pbc, rc, use_cell=True, want_d=True)
        assert np.array_equal(nb, nc) and np.array_equal(lb, lc) and np.array_equal(db, dc)


def test_cell_list_equals_brute_force_open_boundaries_and_unwrapped_positions():
    w = wl.config1(seed=3, cells=7, n_pairs=0)
    pos = w.pos + np.array([[40.0], [-33.0], [5.0]])     # far outside the box on periodic axes
    pbc = np.array([1, 1, 0], dtype=np.int32)
    nb, lb = oracle.neighbors(pos, w.box, pbc, 6.0, use_cell=False)
    nc, lc = oracle.neighbors(pos, w.box, pbc, 6.0, use_cell=True)
    assert np.array_equal(nb, nc) and np.array_equal(lb, lc)
    assert nb.min() < 58 <= nb.max()                     # surface atoms have fewer neighbours


def test_periodic_images_in_a_small_box():
    # one atom in a 5 A cubic box, rc = 6: neighbours are its own images: 6 at 5 A (sqrt(50)=7.07 > 6)
    pos = np.array([[1.0], [2.0], [3.0]])
    nn, nl, nd = oracle.neighbors(pos, np.diag([5.0, 5, 5]).ravel(), [1, 1, 1], 6.0, want_d=True)
    assert nn[0] == 6 and np.all(nl[0, :6] == 0)
    assert sorted(np.linalg.norm(nd[0, :6], axis=1).tolist()) == pytest.approx([5.0] * 6)
    # open in z: only 4 images
    nn, _ = oracle.neighbors(pos, np.diag([5.0, 5, 5]).ravel(), [1, 1, 0], 6.0)
    assert nn[0] == 4


def test_symmetry_of_neighbour_relation():
    w = wl.config1(seed=2, cells=6)
    nn, nl = oracle.neighbors(w.pos, w.box, w.pbc, 5.0)
    S = _sets(nn, nl)
    for i in range(w.n):
        for j in S[i]:
            assert i in S[j]


def test_selection_variant_returns_the_rows_of_the_full_search():
    # orc_neighbors_sel (used by the at-size GPU tests) has no arithmetic of its own: same rows as the brute force
    w = wl.config5(seed=5, cells=(6, 6, 4), vacuum=20.0)
    w.pos = w.pos + wl.rng(5, 21).standard_normal(w.pos.shape) * 0.05
    sel = wl.rng(5, 40).choice(w.n, size=50, replace=False).astype(np.int32)
    for rc in (5.0, 7.0):
        nn, nl = oracle.neighbors(w.pos, w.box, w.pbc, rc, use_cell=False)
        ns, ls = oracle.neighbors(w.pos, w.box, w.pbc, rc, use_cell=True, sel=sel)
        assert np.array_equal(ns, nn[sel]) and np.array_equal(ls, nl[sel])
