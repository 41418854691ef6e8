"""GPU tests of the Wigner-Seitz defect count (ref. [34]; DESIGN C-25) against the
oracle's brute-force nearest-site search: integer results, compared bit for bit."""
import numpy as np
import pytest
import torch

import oracle
from paper_2305_08140_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nb():
    from paper_2305_08140_b200 import binding
    assert torch.cuda.is_available()
    return binding


def _gpu(nb, site, pos, box, pbc):
    g = nb.NepZbl(wl.synthetic_model(), 128)
    g.wigner_seitz_set_reference(torch.from_numpy(np.ascontiguousarray(site)).cuda(), box, pbc)
    nearest, occ, counts = g.wigner_seitz_count(torch.from_numpy(np.ascontiguousarray(pos)).cuda())
    return g, nearest.cpu().numpy(), occ.cpu().numpy(), counts


def test_constructed_defects_bit_exact(nb):
    site, pos, box, pbc, info = wl.defective_lattice(6, seed=2, n_vacancies=5, n_interstitials=3, n_frenkel=4)
    rn, ro, rc = oracle.wigner_seitz(site, pos, box, pbc)
    _, n, o, c = _gpu(nb, site, pos, box, pbc)
    assert np.array_equal(n, rn) and np.array_equal(o, ro) and c == rc == (9, 7)
    assert sorted(np.flatnonzero(o == 0)) == info["vacant"] and sorted(np.flatnonzero(o == 2)) == info["double"]


@pytest.mark.parametrize("pbc", [(1, 1, 1), (1, 1, 0), (0, 0, 0), (0, 1, 0)])
def test_strongly_displaced_atoms_and_open_axes(nb, pbc):
    # sigma = 0.5 A displacements (many atoms leave their cell), ragged cell counts, vacuum on open axes,
    # plus atoms far outside the lattice (sputtered): the ring search must still return the exact nearest site
    site, pos, box, pbc, _ = wl.defective_lattice((5, 6, 7), seed=3, n_vacancies=10, n_interstitials=10,
                                                  n_frenkel=10, sigma=0.5, pbc=pbc, vacuum=15.0)
    g = wl.rng(4, 9)
    far = np.stack([g.uniform(-40.0, 60.0, 40), g.uniform(-40.0, 60.0, 40), g.uniform(-60.0, 90.0, 40)])
    pos = np.ascontiguousarray(np.concatenate([pos, far], axis=1))
    rn, ro, rc = oracle.wigner_seitz(site, pos, box, pbc)
    _, n, o, c = _gpu(nb, site, pos, box, pbc)
    assert np.array_equal(n, rn) and np.array_equal(o, ro) and c == rc


def test_degenerate_inputs(nb):
    a = wl.A0_CONFIG
    site = wl.bcc_lattice(3, 3, 3)
    box = np.diag([3 * a] * 3).ravel()
    h, n, o, c = _gpu(nb, site, np.zeros((3, 0)), box, [1, 1, 1])          # no atoms: every site is vacant
    assert n.size == 0 and np.all(o == 0) and c == (54, 0)
    pos = np.array([[np.nan, 0.1], [0.0, 0.1], [0.0, 0.1]])
    nearest, occ, c = h.wigner_seitz_count(torch.from_numpy(pos).cuda())    # non-finite position: unassigned
    assert nearest.cpu().tolist() == [-1, 0] and c == (53, 0)
    one = np.array([[1.0], [2.0], [3.0]])                                  # a single reference site
    _, n1, o1, c1 = _gpu(nb, one, wl.bcc_lattice(2, 2, 2), box, [1, 1, 0])
    assert np.all(n1 == 0) and o1.tolist() == [16] and c1 == (0, 15)
    g2 = nb.NepZbl(wl.synthetic_model(), 128)
    with pytest.raises(nb.NepZblError):
        g2.wigner_seitz_count(torch.zeros((3, 4), dtype=torch.float64).cuda(), want_occupancy=False)


def test_config2_sized_lattice_sampled(nb):
    # 40^3 cells = 128 000 sites (BASELINE.json configs[1] shape): constructed defects found exactly; nearest
    # site of 1 500 sampled atoms against the oracle's brute force
    site, pos, box, pbc, info = wl.defective_lattice(40, seed=5, n_vacancies=40, n_interstitials=25, n_frenkel=30)
    _, n, o, c = _gpu(nb, site, pos, box, pbc)
    assert c == (70, 55) and o.sum() == pos.shape[1]
    assert sorted(np.flatnonzero(o == 0)) == info["vacant"] and sorted(np.flatnonzero(o == 2)) == info["double"]
    sel = wl.rng(6, 9).choice(pos.shape[1], 1500, replace=False).astype(np.int32)
    rn, _, _ = oracle.wigner_seitz(site, pos, box, pbc, sel=sel)
    assert np.array_equal(n[sel], rn[sel])
    assert np.array_equal(o, np.bincount(n, minlength=site.shape[1]))


def test_foil_sized_lattice_properties(nb):
    # 80 x 80 x 50 cells (640 000 sites), open z with vacuum (configs[4] shape at 1/8 size)
    site, pos, box, pbc, info = wl.defective_lattice((80, 80, 50), seed=7, n_vacancies=100, n_interstitials=60,
                                                     n_frenkel=50, pbc=(1, 1, 0), vacuum=20.0)
    g, n, o, c = _gpu(nb, site, pos, box, pbc)
    assert c == (150, 110) and o.sum() == pos.shape[1] and o.max() == 2
    assert sorted(np.flatnonzero(o == 0)) == info["vacant"] and sorted(np.flatnonzero(o == 2)) == info["double"]
    sel = wl.rng(8, 9).choice(pos.shape[1], 300, replace=False).astype(np.int32)
    rn, _, _ = oracle.wigner_seitz(site, pos, box, pbc, sel=sel)
    assert np.array_equal(n[sel], rn[sel])
    # rerun: identical integers
    n2, o2, c2 = g.wigner_seitz_count(torch.from_numpy(pos).cuda())
    assert np.array_equal(n2.cpu().numpy(), n) and np.array_equal(o2.cpu().numpy(), o) and c2 == c
