"""GPU parity in TRICLINIC boxes (C-28): fractional fixed-point coordinates on the
GPU against the oracle's explicit lattice-vector images."""
import numpy as np
import pytest
import torch

import oracle
from paper_2305_08140_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nb():
    from paper_2305_08140_b200 import binding
    assert torch.cuda.is_available()
    return binding


def _sheared_description(box):
    """(a, b + a, c - a): another cell of the same lattice; its heights are L / sqrt(3) ... L / sqrt(2)."""
    B = box.reshape(3, 3)
    return np.array([B[0], B[1] + B[0], B[2] - B[0]]).ravel()


def _strained(w, seed=3, amp=0.06):
    M = np.eye(3) + amp * wl.rng(seed, 50).uniform(-1, 1, size=(3, 3))
    return (w.pos.T @ M).T.copy(), (w.box.reshape(3, 3) @ M).ravel()


def _check(nb, w, pos, box, label, model=None):
    m = model or w.model
    ref = oracle.compute(oracle.Params(m), pos, w.types, box, w.pbc)
    g = nb.NepZbl(m, w.n)
    e, f, v = g.compute(pos, w.types, box, w.pbc)
    r = parity.compare(e, f, v, ref, label=label)
    assert max(r.values()) <= 1.0, (label, r)
    return g, (e, f, v)


def test_strained_triclinic_crystal_energy_force_virial_and_neighbour_sets(nb):
    w = wl.config1(seed=3, cells=6, n_pairs=3)
    pos, box = _strained(w)
    g, _ = _check(nb, w, pos, box, "triclinic crystal")
    assert g.nep_zbl_last_counts()[0] >= 6                        # the pushed pairs are inside the ZBL range
    g.neighbor_build(torch.from_numpy(pos).cuda(), torch.from_numpy(w.types).cuda(), box, w.pbc)
    for which, rc in ((0, 7.0), (1, 5.0)):
        nn, nl = g.neighbor_get(which)
        bad, dup, _ = parity.compare_neighbor_sets(nn.cpu().numpy(), nl.cpu().numpy(), pos, box, w.pbc, rc, oracle)
        assert not bad and not dup, (which, bad[:5], dup[:5])


def test_same_crystal_in_a_sheared_cell_and_unwrapped_positions(nb):
    w = wl.config1(seed=4, cells=8, n_pairs=2)                   # 25.3 A: the sheared cell's heights stay >= 14 A
    box2 = _sheared_description(w.box)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)      # the orthogonal description
    B = w.box.reshape(3, 3)
    shift = (np.array([2, -3, 1]) @ B)[:, None] + np.array([[0.3], [-0.2], [0.1]])
    for pos in (w.pos, w.pos + shift):
        g = nb.NepZbl(w.model, w.n)
        e, f, v = g.compute(pos, w.types, box2, w.pbc)
        r = parity.compare(e, f, v, ref, label="sheared description")
        assert max(r.values()) <= 1.0, r


def test_block_isolated_in_a_triclinic_box(nb):
    w = wl.config1(seed=5, cells=5, n_pairs=1)
    pos, box = _strained(w, seed=5)
    for name, sl in dict(radial=slice(0, 5), l2=slice(10, 15), l4=slice(20, 25), fourbody=slice(25, 30)).items():
        w0 = np.zeros_like(w.model["w0"]); w0[:, sl] = w.model["w0"][:, sl]
        _check(nb, w, pos, box, f"triclinic, block {name}", model=dict(w.model, w0=w0))


def test_disordered_triclinic_cell_goes_through_the_fp64_pass(nb):
    w = wl.config1(seed=6, cells=5, n_pairs=0, sigma=0.45)        # strongly disordered periodic cell
    pos, box = _strained(w, seed=6)
    g, _ = _check(nb, w, pos, box, "disordered triclinic cell")
    assert g.nep_zbl_last_counts()[1] > 50


def test_paper_sized_model_and_two_types_in_a_triclinic_box(nb):
    wp = wl.config1(seed=7, cells=5, n_pairs=1, model=wl.paper_model())
    pos, box = _strained(wp, seed=7)
    _check(nb, wp, pos, box, "paper-sized model, triclinic")
    wa = wl.config1(seed=8, cells=5, n_pairs=1, model=wl.alloy_model())
    wa.types = wl.random_types(wa.n, 8)
    pos, box = _strained(wa, seed=8)
    _check(nb, wa, pos, box, "two types, triclinic")


def test_md_in_a_triclinic_box_follows_oracle_and_wraps_along_lattice_vectors(nb):
    w = wl.bulk_cascade(6, 300.0, seed=9, n_steps=0, name="tri_md")          # a 300 eV recoil: rebuilds, ZBL
    M = np.eye(3) + 0.05 * wl.rng(9, 50).uniform(-1, 1, size=(3, 3))
    pos0, box = (w.pos.T @ M).T.copy(), (w.box.reshape(3, 3) @ M).ravel()
    n = 60
    opos, ovel, odt, *_ = oracle.md_run(oracle.Params(w.model), pos0, w.vel, w.types, box, w.pbc, n, 1.0, 0.015)
    g = nb.NepZbl(w.model, w.n)
    pos = torch.from_numpy(pos0.copy()).cuda(); vel = torch.from_numpy(w.vel.copy()).cuda()
    g.md_init(pos, vel, torch.from_numpy(w.types).cuda(), box, w.pbc)
    assert g.nep_zbl_uses_graph()
    tr, nreb = g.md_run(n, 1.0, 0.015, want_trace=True)
    assert np.allclose(tr, odt, rtol=1e-6)
    p = pos.cpu().numpy()
    Hi = np.linalg.inv(box.reshape(3, 3))
    d = (p - opos).T @ Hi
    d -= np.round(d)
    assert np.abs(d @ box.reshape(3, 3)).max() < 2e-5
    assert np.abs(vel.cpu().numpy() - ovel).max() < 2e-6
    s = p.T @ Hi
    assert s.min() >= -1e-9 and s.max() < 1 + 1e-9                # wrapped into the cell


def test_triclinic_error_codes(nb):
    w = wl.config1(seed=10, cells=8, n_pairs=0)
    g = nb.NepZbl(w.model, w.n)
    box = _sheared_description(w.box)
    with pytest.raises(nb.NepZblError) as ei:                     # open axis with a non-orthogonal box
        g.compute(w.pos, w.types, box, [1, 1, 0])
    assert ei.value.code == -2
    flat = w.box.reshape(3, 3).copy(); flat[2] = [9.0, 0.0, 9.0]   # cell height along c: 9 A < 14 A
    with pytest.raises(nb.NepZblError) as ei:
        g.compute(w.pos, w.types, flat.ravel(), w.pbc)
    assert ei.value.code == -3
    g.compute(w.pos, w.types, box, w.pbc)                         # the handle is still usable
