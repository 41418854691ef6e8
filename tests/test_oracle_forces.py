"""Pins of the oracle's energy / force / virial evaluation by what the
mathematics fixes: finite differences of the total energy, finite strain, invariances, Eq. 1
additivity.  None of these tests calls the CUDA path."""
import numpy as np
import pytest

import oracle
from paper_2305_08140_b200 import workloads as wl


def _small_periodic(seed=11, cells=3, pairs=1):
    """54-atom cell, box 9.495 A < 2 rc: every pair interacts through several periodic images."""
    return wl.config1(seed=seed, cells=cells, n_pairs=pairs, sigma=0.08)


def _etot(P, w, pos=None, box=None):
    r = oracle.compute(P, w.pos if pos is None else pos, w.types, w.box if box is None else box, w.pbc,
                       use_cell=False, want_force=False, want_virial=False)
    return r.energy.sum()


def test_forces_equal_minus_gradient_all_coordinates():
    w = _small_periodic()
    P = oracle.Params(w.model)
    res = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    i, j = w.info["pairs"][0]
    d = w.pos[:, j] - w.pos[:, i]
    assert 1.0 < np.linalg.norm(d) < 2.0          # a ZBL pair is present
    h = 1e-4                                       # SURVEY 8(c) pins: h = 1e-4 A
    fd = np.zeros_like(res.force)
    for a in range(3):
        for k in range(w.n):
            pp = w.pos.copy(); pp[a, k] += h
            pm = w.pos.copy(); pm[a, k] -= h
            fd[a, k] = -(_etot(P, w, pp) - _etot(P, w, pm)) / (2 * h)
    scale = np.abs(res.force).max()
    # central difference error ~ h^2 F'''/6; 4-point Richardson on the worst coordinate tightens it
    assert np.abs(fd - res.force).max() < 2e-6 * scale
    a, k = np.unravel_index(np.argmax(np.abs(fd - res.force)), fd.shape)
    def fdh(hh):
        pp = w.pos.copy(); pp[a, k] += hh
        pm = w.pos.copy(); pm[a, k] -= hh
        return -(_etot(P, w, pp) - _etot(P, w, pm)) / (2 * hh)
    rich = (4 * fdh(h / 2) - fdh(h)) / 3
    assert rich == pytest.approx(res.force[a, k], rel=1e-7, abs=1e-7 * scale)


def test_zero_net_force_and_symmetric_total_virial():
    w = wl.config1(seed=5, cells=4, n_pairs=2)
    P = oracle.Params(w.model)
    res = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    assert np.abs(res.force.sum(axis=1)).max() < 1e-10
    W = res.virial.sum(axis=1).reshape(3, 3)
    assert W == pytest.approx(W.T, abs=1e-9)


def test_virial_diagonal_by_box_strain():
    # sum_i W_i^{aa} = -dE/d eps_aa under x_a -> (1+eps) x_a, L_a -> (1+eps) L_a
    w = _small_periodic(seed=12)
    P = oracle.Params(w.model)
    res = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    W = res.virial.sum(axis=1)
    e = 1e-6
    for a in range(3):
        def E(eps):
            pos = w.pos.copy(); pos[a] *= (1 + eps)
            box = w.box.copy(); box[4 * a] *= (1 + eps)
            return _etot(P, w, pos, box)
        dE = (E(e) - E(-e)) / (2 * e)
        assert W[4 * a] == pytest.approx(-dE, rel=1e-6)


def test_virial_all_nine_components_by_strain_of_free_cluster():
    w = wl.free_cluster(n=30, seed=3, radius=5.0, min_sep=1.3)
    P = oracle.Params(w.model)
    res = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    nn, _ = oracle.neighbors(w.pos, w.box, w.pbc, 2.0)
    assert nn.sum() > 0                            # cluster has ZBL pairs too
    W = res.virial.sum(axis=1).reshape(3, 3)
    c = w.pos.mean(axis=1, keepdims=True)
    e = 1e-6
    for a in range(3):
        for b in range(3):
            def E(eps):
                M = np.eye(3); M[a, b] += eps
                return _etot(P, w, c + M @ (w.pos - c))
            dE = (E(e) - E(-e)) / (2 * e)
            assert W[a, b] == pytest.approx(-dE, rel=2e-6, abs=1e-6)


def test_translation_invariance_across_periodic_boundary():
    w = wl.config1(seed=6, cells=4, n_pairs=1)
    P = oracle.Params(w.model)
    ref = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    shift = np.array([[3.3], [-7.9], [25.1]])      # moves many atoms across the faces
    L = w.box[[0, 4, 8]][:, None]
    for pos in (w.pos + shift, np.mod(w.pos + shift, L)):
        r = oracle.compute(P, pos, w.types, w.box, w.pbc, use_cell=False)
        assert r.energy == pytest.approx(ref.energy, abs=1e-11)
        assert r.force == pytest.approx(ref.force, abs=1e-9)
        assert r.virial == pytest.approx(ref.virial, abs=1e-9)


def test_lattice_rotation_by_90_degrees():
    w = wl.config1(seed=7, cells=4, n_pairs=1)
    P = oracle.Params(w.model)
    ref = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    L = w.box[0]
    pos = np.stack([L - w.pos[1], w.pos[0], w.pos[2]])           # rotate about z: (x,y) -> (-y,x), shifted into the box
    pos = np.mod(pos, L)
    r = oracle.compute(P, pos, w.types, w.box, w.pbc, use_cell=False)
    assert r.energy == pytest.approx(ref.energy, abs=1e-11)
    assert r.force[0] == pytest.approx(-ref.force[1], abs=1e-9)
    assert r.force[1] == pytest.approx(ref.force[0], abs=1e-9)
    assert r.force[2] == pytest.approx(ref.force[2], abs=1e-9)


def test_arbitrary_rotation_of_free_cluster():
    w = wl.free_cluster(n=25, seed=4, radius=5.0, min_sep=1.3)
    P = oracle.Params(w.model)
    ref = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    R, _ = np.linalg.qr(wl.rng(4, 12).standard_normal((3, 3)))
    c = w.pos.mean(axis=1, keepdims=True)
    r = oracle.compute(P, c + R @ (w.pos - c), w.types, w.box, w.pbc, use_cell=False)
    assert r.energy == pytest.approx(ref.energy, abs=1e-11)
    assert r.force == pytest.approx(R @ ref.force, abs=1e-9)
    Wref = ref.virial.T.reshape(-1, 3, 3)
    Wrot = r.virial.T.reshape(-1, 3, 3)
    assert Wrot == pytest.approx(R @ Wref @ R.T, abs=1e-9)


def test_atom_index_permutation():
    w = wl.config1(seed=8, cells=4, n_pairs=1)
    P = oracle.Params(w.model)
    ref = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    perm = wl.rng(8, 13).permutation(w.n)
    r = oracle.compute(P, w.pos[:, perm], w.types[perm], w.box, w.pbc, use_cell=False)
    assert r.energy == pytest.approx(ref.energy[perm], abs=1e-12)
    assert r.force == pytest.approx(ref.force[:, perm], abs=1e-10)
    assert r.virial == pytest.approx(ref.virial[:, perm], abs=1e-10)


def test_eq1_additivity_nep_plus_zbl():
    w = wl.config1(seed=9, cells=5, n_pairs=3)
    m = w.model
    full = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
    m_nep = dict(m, zbl_enabled=0)
    m_zbl = dict(m, w1=np.zeros_like(m["w1"]), b1=0.0)
    nep = oracle.compute(oracle.Params(m_nep), w.pos, w.types, w.box, w.pbc)
    zbl = oracle.compute(oracle.Params(m_zbl), w.pos, w.types, w.box, w.pbc)
    assert full.energy == pytest.approx(nep.energy + zbl.energy, abs=1e-12)
    assert full.force == pytest.approx(nep.force + zbl.force, abs=1e-10)
    assert full.virial == pytest.approx(nep.virial + zbl.virial, abs=1e-10)
    # ZBL touches only the pushed pairs: 2*n_pairs atoms, each with +1/2 U_ZBL(r)
    touched = np.nonzero(zbl.energy)[0]
    assert sorted(touched) == sorted(a for p in w.info["pairs"] for a in p)
    for (i, j) in w.info["pairs"]:
        r = np.linalg.norm(w.pos[:, j] - w.pos[:, i])
        u, _ = oracle.zbl_pair(oracle.Params(m), r)
        assert zbl.energy[i] == pytest.approx(0.5 * u, rel=1e-13)
        assert zbl.energy[j] == pytest.approx(0.5 * u, rel=1e-13)


def test_zbl_is_exactly_zero_on_a_thermal_lattice():
    # "outer cutoff significantly shorter than the nearest-neighbour distance"
    w = wl.thermal_bulk(4, seed=3, sigma_pos=0.05)
    m = w.model
    a = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
    b = oracle.compute(oracle.Params(dict(m, zbl_enabled=0)), w.pos, w.types, w.box, w.pbc)
    assert np.array_equal(a.energy, b.energy) and np.array_equal(a.force, b.force)


def test_perfect_lattice_has_zero_forces_and_equal_site_energies():
    w = wl.thermal_bulk(4, seed=3)
    r = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)
    assert np.abs(r.force).max() < 1e-10
    assert np.ptp(r.energy) < 1e-12


def test_subset_evaluation_matches_full_evaluation():
    w = wl.config1(seed=10, cells=6, n_pairs=2)
    P = oracle.Params(w.model)
    full = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=True)
    sel = np.array([0, 17, 101, 333, w.info["pairs"][0][0], w.info["pairs"][1][1]], dtype=np.int32)
    sub = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=True, sel=sel)
    assert np.array_equal(sub.energy[sel], full.energy[sel])
    assert sub.force[:, sel] == pytest.approx(full.force[:, sel], abs=1e-11)
    assert sub.virial[:, sel] == pytest.approx(full.virial[:, sel], abs=1e-11)
    others = np.setdiff1d(np.arange(w.n), sel)
    assert np.all(np.isnan(sub.energy[others]))


def test_block_isolated_forces_are_all_significant():
    """with the block q_scaler every descriptor block must move forces well above
    the 1e-4 eV/A parity tolerance, otherwise a bug in that block could pass the GPU parity test."""
    w = wl.config1(seed=1, cells=5, n_pairs=0)
    m = w.model
    D = 30
    blocks = dict(radial=slice(0, 5), l1=slice(5, 10), l2=slice(10, 15), l3=slice(15, 20),
                  l4=slice(20, 25), fourbody=slice(25, 30))
    for name, sl in blocks.items():
        w0 = np.zeros_like(m["w0"]); w0[:, sl] = m["w0"][:, sl]
        r = oracle.compute(oracle.Params(dict(m, w0=w0, zbl_enabled=0)), w.pos, w.types, w.box, w.pbc,
                           want_virial=False)
        rms = np.sqrt((r.force ** 2).mean())
        assert rms > 1e-2, (name, rms)


# ------------------------------------------------------------------ two atom types

def _alloy(seed=13, cells=3):
    w = wl.config1(seed=seed, cells=cells, n_pairs=1, sigma=0.08, model=wl.alloy_model())
    w.types = wl.random_types(w.n, seed)
    return w


def test_two_types_forces_equal_minus_gradient():
    w = _alloy()
    assert 0 < w.types.sum() < w.n
    P = oracle.Params(w.model)
    res = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    h = 1e-4
    scale = np.abs(res.force).max()
    i, j = w.info["pairs"][0]
    for k in [i, j] + list(range(0, w.n, 7)):
        for a in range(3):
            pp = w.pos.copy(); pp[a, k] += h
            pm = w.pos.copy(); pm[a, k] -= h
            fd = -(_etot(P, w, pp) - _etot(P, w, pm)) / (2 * h)
            assert fd == pytest.approx(res.force[a, k], abs=2e-6 * scale), (a, k)
    assert np.abs(res.force.sum(axis=1)).max() < 1e-9 * scale * w.n


def test_two_types_reduce_to_one_type_and_relabel():
    w = _alloy(seed=14)
    one = wl.synthetic_model()
    # identical tables / Z / mass for every type pair: the labels cannot matter
    same = dict(one, n_types=2)
    same["c_radial"] = np.broadcast_to(one["c_radial"][0, 0], (2, 2) + one["c_radial"].shape[2:]).copy()
    same["c_angular"] = np.broadcast_to(one["c_angular"][0, 0], (2, 2) + one["c_angular"].shape[2:]).copy()
    same["atomic_number"] = np.array([wl.W_Z, wl.W_Z]); same["mass"] = np.array([wl.W_MASS, wl.W_MASS])
    a = oracle.compute(oracle.Params(same), w.pos, w.types, w.box, w.pbc, use_cell=False)
    b = oracle.compute(oracle.Params(one), w.pos, np.zeros_like(w.types), w.box, w.pbc, use_cell=False)
    assert np.allclose(a.energy, b.energy, rtol=0, atol=1e-12) and np.allclose(a.force, b.force, rtol=0, atol=1e-11)
    # swapping the labels 0 <-> 1 together with every per-type table is the same physical system
    m = w.model
    sw = dict(m, c_radial=m["c_radial"][::-1, ::-1].copy(), c_angular=m["c_angular"][::-1, ::-1].copy(),
              atomic_number=m["atomic_number"][::-1].copy(), mass=m["mass"][::-1].copy())
    c = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc, use_cell=False)
    d = oracle.compute(oracle.Params(sw), w.pos, 1 - w.types, w.box, w.pbc, use_cell=False)
    assert np.allclose(c.energy, d.energy, rtol=0, atol=1e-12) and np.allclose(c.virial, d.virial, rtol=0, atol=1e-10)
    # and the two types really differ: the unswapped labels give other energies
    e = oracle.compute(oracle.Params(m), w.pos, 1 - w.types, w.box, w.pbc, use_cell=False)
    assert np.abs(e.energy - c.energy).max() > 1e-3


def test_five_body_model_forces_and_virial_by_finite_differences():
    # SURVEY 8(f) NEXT-4 / DESIGN C-27: the model with the (1,1,1,1) term, all 3N coordinates and the strain virial
    w = wl.config1(seed=13, cells=3, n_pairs=1, sigma=0.08, model=wl.synthetic_model(has_5body=1))
    P = oracle.Params(w.model)
    res = oracle.compute(P, w.pos, w.types, w.box, w.pbc, use_cell=False)
    h = 1e-4
    fd = np.zeros_like(res.force)
    for a in range(3):
        for k in range(w.n):
            pp = w.pos.copy(); pp[a, k] += h
            pm = w.pos.copy(); pm[a, k] -= h
            fd[a, k] = -(_etot(P, w, pp) - _etot(P, w, pm)) / (2 * h)
    assert np.abs(fd - res.force).max() < 2e-6 * np.abs(res.force).max()
    W = res.virial.sum(axis=1)
    e = 1e-6
    for a in range(3):
        def E(eps):
            pos = w.pos.copy(); pos[a] *= (1 + eps)
            box = w.box.copy(); box[4 * a] *= (1 + eps)
            return _etot(P, w, pos, box)
        assert W[4 * a] == pytest.approx(-(E(e) - E(-e)) / (2 * e), rel=1e-6)
    # the block matters: zeroing its W0 columns changes the energies
    m0 = dict(w.model); w0 = m0["w0"].copy(); w0[:, 30:] = 0.0; m0["w0"] = w0
    r0 = oracle.compute(oracle.Params(m0), w.pos, w.types, w.box, w.pbc, use_cell=False, want_force=False, want_virial=False)
    assert np.abs(r0.energy - res.energy).max() > 1e-3
