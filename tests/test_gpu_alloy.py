"""GPU parity with two atom types (the type-pair coefficient tables c^{ti tj}_nk, per-type atomic
numbers in the ZBL term and per-type masses in the integrator are exercised) against the fp64 oracle."""
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


def _alloy(seed=1, cells=6, n_pairs=3):
    w = wl.config1(seed=seed, cells=cells, n_pairs=n_pairs, model=wl.alloy_model())
    w.types = wl.random_types(w.n, seed)
    return w


def test_energy_force_virial_descriptors(nb):
    w = _alloy()
    # the pushed pairs cover W-W, W-Mo or Mo-Mo contacts: the ZBL term sees both atomic numbers
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, want_q=True)
    g = nb.NepZbl(w.model, w.n)
    e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
    r = parity.compare(e, f, v, ref, label="two types")
    assert max(r.values()) <= 1.0, r
    q = g.nep_zbl_get_descriptors().cpu().numpy()
    scale = np.asarray(w.model["q_scaler"])
    err = np.abs(q - ref.q) * scale
    assert (err / (2e-5 + 3e-6 * np.abs(ref.q * scale))).max() < 1.0
    zi = [a for p in w.info["pairs"] for a in p]
    assert ref.energy[zi].max() > 1.0
    # the labels matter: the same positions with all atoms of type 0 give other energies
    e0, _, _ = nb.NepZbl(w.model, w.n).compute(w.pos, np.zeros_like(w.types), w.box, w.pbc)
    assert np.abs(e0 - e).max() > 1e-2


def test_block_isolated(nb):
    w = _alloy(seed=2, cells=5, n_pairs=1)
    blocks = dict(radial=slice(0, 5), l1=slice(5, 10), l2=slice(10, 15), l3=slice(15, 20), l4=slice(20, 25),
                  fourbody=slice(25, 30))
    for name, sl in blocks.items():
        w0 = np.zeros_like(w.model["w0"]); w0[:, sl] = w.model["w0"][:, sl]
        m = dict(w.model, w0=w0)
        ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
        e, f, v = nb.NepZbl(m, w.n).compute(w.pos, w.types, w.box, w.pbc)
        r = parity.compare(e, f, v, ref, label=f"two types, block {name}")
        assert max(r.values()) <= 1.0, (name, r)


def test_identical_tables_reduce_to_one_type(nb):
    w = _alloy(seed=3, cells=5, n_pairs=2)
    one = wl.synthetic_model()
    same = dict(one, n_types=2)
    same["c_radial"] = np.broadcast_to(one["c_radial"][0, 0], (2, 2) + one["c_radial"].shape[2:]).copy()
    same["c_angular"] = np.broadcast_to(one["c_angular"][0, 0], (2, 2) + one["c_angular"].shape[2:]).copy()
    same["atomic_number"] = np.array([wl.W_Z, wl.W_Z]); same["mass"] = np.array([wl.W_MASS, wl.W_MASS])
    e2, f2, v2 = nb.NepZbl(same, w.n).compute(w.pos, w.types, w.box, w.pbc)
    e1, f1, v1 = nb.NepZbl(one, w.n).compute(w.pos, np.zeros_like(w.types), w.box, w.pbc)
    # two fp32 code paths for the same numbers (the one-type kernels read {rhat, r} per angular neighbour, the two-type
    # kernels {d, type}): they agree to a few fp32 ulp of the ~10 eV site energies, half the oracle tolerance at most
    assert np.abs(e2 - e1).max() < 5e-6 and np.abs(f2 - f1).max() < 2e-4 * max(1.0, np.abs(f1).max() * 1e-2)


def test_md_with_two_masses_follows_oracle(nb):
    w = wl.thermal_bulk(6, seed=4, sigma_pos=0.03, model=wl.alloy_model())
    w.types = wl.random_types(w.n, 4)
    P = oracle.Params(w.model)
    n = 30
    opos, ovel, odt, oep, oek = oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, n, 1.0, 0.01)
    g = nb.NepZbl(w.model, w.n)
    pos = torch.from_numpy(w.pos.copy()).cuda(); vel = torch.from_numpy(w.vel.copy()).cuda()
    g.md_init(pos, vel, torch.from_numpy(w.types).cuda(), w.box, w.pbc)
    tr, _ = g.md_run(n, 1.0, 0.01, want_trace=True)
    L = w.box[[0, 4, 8]][:, None]
    d = pos.cpu().numpy() - opos
    d -= L * np.round(d / L)
    assert np.allclose(tr, odt, rtol=1e-6)
    assert np.abs(d).max() < 5e-6 and np.abs(vel.cpu().numpy() - ovel).max() < 5e-7
    ep, ek = g.md_energies()
    assert ep == pytest.approx(oep[-1], abs=2e-5 * w.n) and ek == pytest.approx(oek[-1], rel=1e-4)
