"""GPU parity for the rest of SURVEY 8(f) NEXT-4 ("high-entropy alloys" -- NEP generality): the 5-body
(1,1,1,1) term (C-27) and two atom types at the PAPER-sized model shape (n_max 15 / 10, 100 neurons,
P:106), against the fp64 oracle at the north_star tolerances."""
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


def _check(nb, w, label, model=None, use_cell=None):
    m = model or w.model
    ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc, use_cell=use_cell)
    g = nb.NepZbl(m, w.n)
    e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
    r = parity.compare(e, f, v, ref, label=label)
    assert max(r.values()) <= 1.0, (label, r)
    return g


# ------------------------------------------------------------------ 5-body term

def test_five_body_model_energy_force_virial_descriptors(nb):
    m = wl.synthetic_model(has_5body=1)
    w = wl.config1(seed=1, cells=6, n_pairs=2, model=m)
    assert oracle.Params(m).D == 35
    g = _check(nb, w, "5-body model")
    ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc, want_q=True, want_force=False, want_virial=False)
    q = g.nep_zbl_get_descriptors().cpu().numpy()
    s = np.asarray(m["q_scaler"])
    # atoms on the fp32 path: absolute error in network-input units; listed atoms: fp64 values rounded to fp32
    err = np.abs(q - ref.q) * s
    assert (err / (2e-5 + 3e-6 * np.abs(ref.q * s))).max() < 1.0
    assert np.abs(ref.q[:, 30:] * s[30:]).max() > 1.0            # the block is alive


def test_five_body_block_isolated_and_on_a_cluster(nb):
    m = wl.synthetic_model(has_5body=1)
    w = wl.config1(seed=2, cells=5, n_pairs=1, model=m)
    w0 = np.zeros_like(m["w0"]); w0[:, 30:] = m["w0"][:, 30:]
    _check(nb, w, "5-body block alone", model=dict(m, w0=w0))
    w0 = np.zeros_like(m["w0"]); w0[:, 5:10] = m["w0"][:, 5:10]; w0[:, 30:] = m["w0"][:, 30:]
    _check(nb, w, "l = 1 and 5-body blocks (they share A_1m)", model=dict(m, w0=w0))
    wc = wl.free_cluster(n=50, seed=16, radius=6.0, min_sep=1.4, model=m)      # disordered: the fp64 pass carries the term
    g = _check(nb, wc, "5-body model, random cluster", use_cell=False)
    assert g.nep_zbl_last_counts()[1] > 20


def test_five_body_md_follows_oracle(nb):
    m = wl.synthetic_model(has_5body=1)
    w = wl.thermal_bulk(5, seed=3, sigma_pos=0.03, model=m)
    n = 20
    opos, ovel, odt, oep, oek = oracle.md_run(oracle.Params(m), w.pos, w.vel, w.types, w.box, w.pbc, n, 1.0, 0.01)
    g = nb.NepZbl(m, w.n)
    pos = torch.from_numpy(w.pos.copy()).cuda(); vel = torch.from_numpy(w.vel.copy()).cuda()
    g.md_init(pos, vel, torch.from_numpy(w.types).cuda(), w.box, w.pbc)
    g.md_run(n, 1.0, 0.01)
    L = w.box[[0, 4, 8]][:, None]
    d = pos.cpu().numpy() - opos
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 5e-6 and np.abs(vel.cpu().numpy() - ovel).max() < 5e-7


# ------------------------------------------------------------------ two atom types, paper-sized model

def _paper_alloy(spread=0.3):
    one = wl.paper_model()
    m = dict(one, n_types=2)
    g = wl.rng(184, 17)
    for key in ("c_radial", "c_angular"):       # the recipe of workloads.alloy_model on the paper-sized tables
        c = np.broadcast_to(one[key][0, 0], (2, 2) + one[key].shape[2:])
        m[key] = c * (1.0 + spread * g.uniform(-1.0, 1.0, size=c.shape))
    m["atomic_number"] = np.array([wl.W_Z, wl.MO_Z]); m["mass"] = np.array([wl.W_MASS, wl.MO_MASS])
    return m


def test_paper_sized_two_types_energy_force_virial(nb):
    m = _paper_alloy()
    w = wl.config1(seed=4, cells=6, n_pairs=3, model=m)
    w.types = wl.random_types(w.n, 4)
    g = _check(nb, w, "paper-sized model, two types")
    # the labels matter
    e, _, _ = g.compute(w.pos, w.types, w.box, w.pbc)
    e0, _, _ = nb.NepZbl(m, w.n).compute(w.pos, np.zeros_like(w.types), w.box, w.pbc)
    assert np.abs(e0 - e).max() > 1e-2


def test_paper_sized_two_types_block_isolated_and_cluster(nb):
    m = _paper_alloy()
    w = wl.config1(seed=5, cells=5, n_pairs=1, model=m)
    w.types = wl.random_types(w.n, 5)
    NR, NA = 16, 11
    for name, sl in dict(radial=slice(0, NR), l1=slice(NR, NR + NA), l3=slice(NR + 2 * NA, NR + 3 * NA),
                         l4=slice(NR + 3 * NA, NR + 4 * NA)).items():
        w0 = np.zeros_like(m["w0"]); w0[:, sl] = m["w0"][:, sl]
        _check(nb, w, f"paper-sized two types, block {name}", model=dict(m, w0=w0))
    wc = wl.free_cluster(n=45, seed=17, radius=6.0, min_sep=1.5, model=m)
    wc.types = wl.random_types(wc.n, 17)
    _check(nb, wc, "paper-sized two types, random cluster", use_cell=False)


def test_paper_sized_identical_tables_reduce_to_one_type(nb):
    one = wl.paper_model()
    same = dict(one, n_types=2)
    same["c_radial"] = np.broadcast_to(one["c_radial"][0, 0], (2, 2) + one["c_radial"].shape[2:]).copy()
    same["c_angular"] = np.broadcast_to(one["c_angular"][0, 0], (2, 2) + one["c_angular"].shape[2:]).copy()
    same["atomic_number"] = np.array([wl.W_Z, wl.W_Z]); same["mass"] = np.array([wl.W_MASS, wl.W_MASS])
    w = wl.config1(seed=6, cells=5, n_pairs=2, model=one)
    types = wl.random_types(w.n, 6)
    e2, f2, v2 = nb.NepZbl(same, w.n).compute(w.pos, types, w.box, w.pbc)
    e1, f1, v1 = nb.NepZbl(one, w.n).compute(w.pos, np.zeros_like(types), w.box, w.pbc)
    # two fp32 code paths for the same numbers (the one-type kernels read {rhat, r} per angular neighbour, the two-type
    # kernels {d, type}): they agree to a few fp32 ulp of the ~10 eV site energies, half the oracle tolerance at most
    assert np.abs(e2 - e1).max() < 5e-6 and np.abs(f2 - f1).max() < 2e-4 * max(1.0, np.abs(f1).max() * 1e-2)


def test_paper_sized_two_types_md_follows_oracle(nb):
    m = _paper_alloy(spread=0.05)
    w = wl.thermal_bulk(5, seed=7, sigma_pos=0.03, model=m, a=wl.A0_PAPER)
    w.types = wl.random_types(w.n, 7)
    n = 20
    opos, ovel, *_ = oracle.md_run(oracle.Params(m), w.pos, w.vel, w.types, w.box, w.pbc, n, 1.0, 0.01)
    g = nb.NepZbl(m, w.n)
    pos = torch.from_numpy(w.pos.copy()).cuda(); vel = torch.from_numpy(w.vel.copy()).cuda()
    g.md_init(pos, vel, torch.from_numpy(w.types).cuda(), w.box, w.pbc)
    g.md_run(n, 1.0, 0.01)
    L = w.box[[0, 4, 8]][:, None]
    d = pos.cpu().numpy() - opos
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 5e-6 and np.abs(vel.cpu().numpy() - ovel).max() < 5e-7
