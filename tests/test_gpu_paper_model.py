"""GPU parity for the paper-sized model (sizes P:106, ZBL refit Eq. 3): the
four-lanes-per-atom kernel k_angular_nn_split against the fp64 oracle at the north_star tolerances."""
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


def _case(seed=1, cells=6, n_pairs=3):
    return wl.config1(seed=seed, cells=cells, n_pairs=n_pairs, model=wl.paper_model())


def test_energy_force_virial_and_descriptors(nb):
    w = _case()
    assert oracle.Params(w.model).D == 60
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, want_q=True)
    g = nb.NepZbl(w.model, w.n)
    e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
    r = parity.compare(e, f, v, ref, label="paper model")
    assert max(r.values()) <= 1.0, r
    q = g.nep_zbl_get_descriptors().cpu().numpy()
    scale = np.asarray(w.model["q_scaler"])
    err = np.abs(q - ref.q) * scale
    assert (err / (2e-5 + 3e-6 * np.abs(ref.q * scale))).max() < 1.0
    zi = [a for p in w.info["pairs"] for a in p]
    assert ref.energy[zi].max() > 1.0      # ZBL (Eq. 3 refit) is active on the pushed pairs


def test_block_isolated(nb):
    # every descriptor block alone drives the network: a bug confined to one block cannot hide
    w = _case(seed=2, cells=5, n_pairs=1)
    NR, NA = 16, 11
    blocks = dict(radial=slice(0, NR), l1=slice(NR, NR + NA), l2=slice(NR + NA, NR + 2 * NA),
                  l3=slice(NR + 2 * NA, NR + 3 * NA), l4=slice(NR + 3 * NA, NR + 4 * NA))
    for name, sl in blocks.items():
        w0 = np.zeros_like(w.model["w0"]); w0[:, sl] = w.model["w0"][:, sl]
        m = dict(w.model, w0=w0)
        ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
        g = nb.NepZbl(m, w.n)
        e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
        r = parity.compare(e, f, v, ref, label=f"paper model, block {name}")
        assert max(r.values()) <= 1.0, (name, r)


def test_ragged_sizes_and_determinism(nb):
    # n not a multiple of 8 (atoms per warp): a free cluster of 45 atoms in an open box
    w = wl.free_cluster(n=45, seed=9, radius=8.0, min_sep=2.2, model=wl.paper_model())
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)
    outs = []
    for _ in range(2):
        g = nb.NepZbl(w.model, w.n)
        outs.append(g.compute(w.pos, w.types, w.box, w.pbc))
    r = parity.compare(*outs[0], ref, label="paper model, cluster")
    assert max(r.values()) <= 1.0, r
    for a, b in zip(outs[0], outs[1]):
        assert a.tobytes() == b.tobytes()


def test_md_follows_oracle(nb):
    w = wl.paper_bulk(5, seed=3, sigma_pos=0.03)
    P = oracle.Params(w.model)
    n = 20
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


def test_bench_sized_system_sampled(nb):
    # the system bench.py --workload paper times (40^3 cells, 128 000 atoms), positions displaced by 0.05 A:
    # 512 sampled atoms against the oracle, which evaluates them one by one
    w = wl.paper_bulk(40, seed=12)
    w.pos = np.mod(w.pos + wl.rng(12, 23).standard_normal(w.pos.shape) * 0.05, w.box[[0, 4, 8]][:, None])
    g = nb.NepZbl(w.model, w.n)
    e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
    sel = np.sort(wl.rng(12, 24).choice(w.n, size=512, replace=False)).astype(np.int32)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, sel=sel)
    r = parity.compare(e, f, v, ref, idx=sel, label="paper model, 128 000 atoms, sample")
    assert max(r.values()) <= 1.0, r
    assert np.abs(f.sum(axis=1)).max() < 0.1


def test_both_network_paths(nb, monkeypatch):
    """The four-lane kernel has two forms: k_angular_split_tc (network on the tensor cores, the default here) and
    k_angular_nn_split (FFMA network; more than 104 neurons, cap_angular > 64, NEPZBL_NN=ffma).  Both against the oracle."""
    w = _case(seed=3, cells=5, n_pairs=2)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)
    g = nb.NepZbl(w.model, w.n)
    assert g.nep_zbl_network_mode() == 3
    r = parity.compare(*g.compute(w.pos, w.types, w.box, w.pbc), ref, label="paper model, tensor-core network")
    assert max(r.values()) <= 1.0, r
    monkeypatch.setenv("NEPZBL_NN", "ffma")
    g = nb.NepZbl(w.model, w.n)
    assert g.nep_zbl_network_mode() == 0
    r = parity.compare(*g.compute(w.pos, w.types, w.box, w.pbc), ref, label="paper model, FFMA network")
    assert max(r.values()) <= 1.0, r
    monkeypatch.delenv("NEPZBL_NN")
    big = wl.paper_model()
    big = dict(big, n_neurons=120, w0=np.vstack([big["w0"], big["w0"][:20] * 0.5]), b0=np.concatenate([big["b0"], big["b0"][:20]]),
               w1=np.concatenate([big["w1"], big["w1"][:20] * 0.1]))
    g = nb.NepZbl(big, w.n)
    assert g.nep_zbl_network_mode() == 0       # 120 neurons: beyond the tensor-core form, same results path
    ref = oracle.compute(oracle.Params(big), w.pos, w.types, w.box, w.pbc)
    r = parity.compare(*g.compute(w.pos, w.types, w.box, w.pbc), ref, label="paper model, 120 neurons")
    assert max(r.values()) <= 1.0, r
