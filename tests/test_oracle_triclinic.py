"""Pins of the oracle's triclinic boxes (C-28): lattice-vector images instead of
per-axis shifts.  What fixes it from outside: the SAME infinite crystal described by a different (sheared) cell, a
rigid rotation of cell and atoms, an explicit supercell without periodicity, finite differences and cell strain."""
import numpy as np
import pytest

import oracle
from paper_2305_08140_b200 import workloads as wl


def _sheared_description(w):
    """Lattice vectors (a, b + a, c + 2a - b): another unit cell of the same lattice (unimodular combination)."""
    B = w.box.reshape(3, 3)
    return np.array([B[0], B[1] + B[0], B[2] + 2 * B[0] - B[1]]).ravel()


def _strained(w, seed=3, amp=0.06):
    """A genuinely triclinic crystal: homogeneous deformation x -> x M of cell and atoms (M = 1 + small random)."""
    M = np.eye(3) + amp * wl.rng(seed, 50).uniform(-1, 1, size=(3, 3))
    box = (w.box.reshape(3, 3) @ M).ravel()
    pos = (w.pos.T @ M).T.copy()
    return pos, box


def test_same_crystal_other_cell_gives_the_same_results():
    w = wl.config1(seed=3, cells=5, n_pairs=1)
    P = oracle.Params(w.model)
    ref = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    r = oracle.compute(P, w.pos, w.types, _sheared_description(w), w.pbc)
    assert r.energy == pytest.approx(ref.energy, abs=1e-11)
    assert r.force == pytest.approx(ref.force, abs=1e-10)
    assert r.virial == pytest.approx(ref.virial, abs=1e-10)
    # positions given far outside the cell are wrapped along the lattice vectors
    B = w.box.reshape(3, 3)
    shift = (np.array([3, -2, 5]) @ B)[:, None] + 0.0
    r2 = oracle.compute(P, w.pos + shift, w.types, _sheared_description(w), w.pbc)
    assert r2.energy == pytest.approx(ref.energy, abs=1e-10) and r2.force == pytest.approx(ref.force, abs=1e-9)


def test_rigid_rotation_of_cell_and_atoms():
    w = wl.config1(seed=4, cells=5, n_pairs=1)
    P = oracle.Params(w.model)
    ref = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    R, _ = np.linalg.qr(wl.rng(4, 51).standard_normal((3, 3)))
    if np.linalg.det(R) < 0:
        R[:, 0] *= -1
    box = (w.box.reshape(3, 3) @ R.T).ravel()              # rows (lattice vectors) rotated
    pos = R @ w.pos
    r = oracle.compute(P, pos, w.types, box, w.pbc)
    assert r.energy == pytest.approx(ref.energy, abs=1e-11)
    assert r.force == pytest.approx(R @ ref.force, abs=1e-10)
    Wref = ref.virial.reshape(3, 3, -1)
    Wrot = np.einsum("ab,bcn,dc->adn", R, Wref, R)
    assert r.virial.reshape(3, 3, -1) == pytest.approx(Wrot, abs=1e-10)


def test_neighbours_against_an_explicit_supercell():
    w = wl.config1(seed=5, cells=4, n_pairs=0)
    pos, box = _strained(w)
    rc = 6.0
    nn, nl, nd = oracle.neighbors(pos, box, w.pbc, rc, want_d=True)
    B = box.reshape(3, 3)
    # explicit 5x5x5 supercell (|s| <= 2 covers rc = 6 A for cell heights ~12 A), plain distances, no periodicity
    Hi = np.linalg.inv(B)
    s = pos.T @ Hi
    pw = ((s - np.floor(s)) @ B)                                              # (n, 3) wrapped
    shifts = np.array([[i, j, k] for i in range(-2, 3) for j in range(-2, 3) for k in range(-2, 3)]) @ B
    for i in range(0, w.n, 7):
        d = (pw[None, :, :] + shifts[:, None, :]) - pw[i]                      # (125, n, 3)
        r = np.linalg.norm(d, axis=2)
        hit = (r < rc) & (r > 0)
        assert nn[i] == hit.sum()
        got = sorted(np.round(np.linalg.norm(nd[i, :nn[i]], axis=1), 9).tolist())
        assert got == sorted(np.round(r[hit], 9).tolist())


def test_forces_and_full_virial_of_a_triclinic_crystal_by_finite_differences():
    w = wl.config1(seed=6, cells=3, n_pairs=1, sigma=0.08)
    pos, box = _strained(w)
    P = oracle.Params(w.model)

    def etot(p, b):
        return oracle.compute(P, p, w.types, b, w.pbc, want_force=False, want_virial=False).energy.sum()

    res = oracle.compute(P, pos, w.types, box, w.pbc)
    assert np.abs(res.force.sum(axis=1)).max() < 1e-10
    h = 1e-4
    fd = np.zeros_like(res.force)
    for a in range(3):
        for k in range(w.n):
            pp = pos.copy(); pp[a, k] += h
            pm = pos.copy(); pm[a, k] -= h
            fd[a, k] = -(etot(pp, box) - etot(pm, box)) / (2 * h)
    assert np.abs(fd - res.force).max() < 2e-6 * np.abs(res.force).max()
    # all nine components: x -> x (1 + eps e_a e_b^T) applied to cell rows and atoms; sum_i W_i^{ab} = -dE/d eps_ab
    W = res.virial.sum(axis=1).reshape(3, 3)
    assert W == pytest.approx(W.T, abs=1e-8)
    e = 1e-6
    for a in range(3):
        for b in range(3):
            def E(eps):
                M = np.eye(3); M[a, b] += eps
                return etot(M @ pos, (box.reshape(3, 3) @ M.T).ravel())
            assert W[a, b] == pytest.approx(-(E(e) - E(-e)) / (2 * e), rel=2e-6, abs=1e-6)


def test_md_in_the_sheared_description_follows_the_orthogonal_one():
    w = wl.thermal_bulk(5, seed=7, sigma_pos=0.03)
    P = oracle.Params(w.model)
    n = 25
    p1, v1, dt1, ep1, ek1 = oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, n, 1.0, 0.01, use_cell=False)
    box2 = _sheared_description(w)
    p2, v2, dt2, ep2, ek2 = oracle.md_run(P, w.pos, w.vel, w.types, box2, w.pbc, n, 1.0, 0.01)
    assert dt2 == pytest.approx(dt1, rel=1e-12)
    assert v2 == pytest.approx(v1, abs=1e-12)
    d = (p2 - p1).T @ np.linalg.inv(w.box.reshape(3, 3))                      # differ by lattice vectors only
    assert np.abs(d - np.round(d)).max() < 1e-10
    assert ep2 == pytest.approx(ep1, abs=1e-9)
    # wrapped into the sheared cell: fractional coordinates in [0, 1)
    s = p2.T @ np.linalg.inv(box2.reshape(3, 3))
    assert s.min() >= -1e-12 and s.max() < 1 + 1e-12


def test_open_axes_are_refused_for_triclinic_boxes():
    w = wl.config1(seed=8, cells=4, n_pairs=0)
    with pytest.raises(RuntimeError):
        oracle.compute(oracle.Params(w.model), w.pos, w.types, _sheared_description(w), [1, 1, 0])
