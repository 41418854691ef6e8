"""GPU parity on DISORDERED sites -- random clusters and the molten core of a cascade, the close encounters the
paper's ZBL term exists for -- at the SAME north_star tolerances as the lattice-like cases.

On such sites the angular network inputs s_nu q_nu are 10-1000x their lattice values and an fp32 evaluation misses
the tolerances by up to 2.7x (only the 4-body block fails when the blocks are isolated;
test_fp32_alone_misses_the_tolerance below keeps that measurement).  The library lists every atom with an angular input above its threshold and re-evaluates it in
fp64 (csrc/site_fp64.cuh).  These tests hold every case to 1.0 x the tolerance and check that the fp64 pass really
ran here and did NOT run on a thermal crystal."""
import numpy as np
import pytest
import torch

import oracle
from paper_2305_08140_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

BLOCKS = dict(radial=slice(0, 5), l1=slice(5, 10), l2=slice(10, 15), l3=slice(15, 20), l4=slice(20, 25),
              fourbody=slice(25, 30))


@pytest.fixture(scope="module")
def nb():
    from paper_2305_08140_b200 import binding
    assert torch.cuda.is_available()
    return binding


def _check(nb, w, label, model=None):
    m = model or w.model
    ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc, use_cell=False)
    g = nb.NepZbl(m, w.n)
    e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
    r = parity.compare(e, f, v, ref, label=label)
    assert max(r.values()) <= 1.0, (label, r)
    return g, (e, f, v)


@pytest.mark.parametrize("kw", [dict(n=60, seed=8, radius=7.0, min_sep=1.7),     # round 1's 5x case
                                dict(n=60, seed=7, radius=6.0, min_sep=1.3),     # the case commit d2c5db4 dropped
                                dict(n=60, seed=8, radius=6.0, min_sep=1.3),
                                dict(n=97, seed=21, radius=7.5, min_sep=1.1)])
def test_random_cluster_at_the_stated_tolerance(nb, kw):
    w = wl.free_cluster(**kw)
    g, _ = _check(nb, w, f"random cluster {kw}")
    n_zbl, n_fp64 = g.nep_zbl_last_counts()
    assert n_fp64 > w.n // 2          # disordered: almost every atom goes through the fp64 pass
    assert n_zbl > 0                  # and pairs inside 2 A are present


def test_random_cluster_block_isolated(nb):
    """SURVEY 8(c) C-6 on a disordered cluster: with only one descriptor block driving the network a bug (or a
    precision loss) confined to that block cannot hide behind the others."""
    w = wl.free_cluster(n=60, seed=8, radius=6.0, min_sep=1.3)
    for name, sl in BLOCKS.items():
        w0 = np.zeros_like(w.model["w0"]); w0[:, sl] = w.model["w0"][:, sl]
        _check(nb, w, f"random cluster, block {name}", model=dict(w.model, w0=w0))


def test_fp64_pass_descriptors_and_determinism(nb):
    w = wl.free_cluster(n=60, seed=8, radius=7.0, min_sep=1.7)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, use_cell=False, want_q=True,
                         want_force=False, want_virial=False)
    outs = []
    for _ in range(3):
        g, out = _check(nb, w, "cluster rerun")
        outs.append(out)
    for o in outs[1:]:     # the fp64 list is filled in ticket order; the results do not depend on it
        for a, b in zip(outs[0], o):
            assert a.tobytes() == b.tobytes()
    # descriptors of the listed atoms come from the fp64 pass: fp32 rounding of the STORED value only
    q = g.nep_zbl_get_descriptors().cpu().numpy()
    s = np.asarray(w.model["q_scaler"])
    ang = slice(5, 30)
    big = np.abs(ref.q[:, 25:30] * s[25:30]).max(axis=1) > 3.5
    assert big.sum() > 30
    rel = np.abs(q[big][:, ang] - ref.q[big][:, ang]) / np.maximum(np.abs(ref.q[big][:, ang]), 1e-30)
    assert rel.max() < 2e-7


def test_fp32_alone_misses_the_tolerance(nb, monkeypatch):
    """The measurement behind the fp64 pass: with the pass switched off (NEPZBL_DENSE_THRESHOLD=off, a measurement
    aid read at create) the fp32 kernels alone exceed the tolerance on these clusters (round 2: 1.55x, 2.39x, 2.66x)
    while config 1 -- lattice-like sites -- passes either way."""
    monkeypatch.setenv("NEPZBL_DENSE_THRESHOLD", "off")
    worst = []
    for kw in (dict(n=60, seed=8, radius=7.0, min_sep=1.7), dict(n=60, seed=7, radius=6.0, min_sep=1.3),
               dict(n=60, seed=8, radius=6.0, min_sep=1.3)):
        w = wl.free_cluster(**kw)
        ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, use_cell=False)
        g = nb.NepZbl(w.model, w.n)
        e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
        assert g.nep_zbl_last_counts()[1] == 0
        worst.append(max(parity.compare(e, f, v, ref, label=f"fp32 only, cluster {kw}").values()))
    assert min(worst) > 1.0 and max(worst) < 5.0, worst
    w = wl.config1()
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)
    e, f, v = nb.NepZbl(w.model, w.n).compute(w.pos, w.types, w.box, w.pbc)
    assert max(parity.compare(e, f, v, ref, label="fp32 only, config1").values()) <= 1.0


def test_thermal_crystal_lists_no_atom(nb):
    w = wl.thermal_bulk(8, seed=5, sigma_pos=0.05)
    g = nb.NepZbl(w.model, w.n)
    g.compute(w.pos, w.types, w.box, w.pbc)
    assert g.nep_zbl_last_counts() == (0, 0)


def test_free_surface_is_not_listed(nb):
    # the atoms of a free (001) surface have large but COHERENT l = 1 sums (accurate in fp32): they stay on the fp32 path
    w = wl.config5(seed=5, cells=(8, 8, 6), vacuum=20.0)
    w.pos = w.pos + wl.rng(5, 21).standard_normal(w.pos.shape) * 0.05
    g, _ = _check(nb, w, "foil surfaces")
    assert g.nep_zbl_last_counts() == (0, 0)


def test_two_types_and_paper_sized_model_on_a_cluster(nb):
    wa = wl.free_cluster(n=50, seed=14, radius=6.0, min_sep=1.4, model=wl.alloy_model())
    wa.types = wl.random_types(wa.n, 14)
    g, _ = _check(nb, wa, "two-type cluster")
    assert g.nep_zbl_last_counts()[1] > 20
    wp = wl.free_cluster(n=45, seed=9, radius=6.0, min_sep=1.5, model=wl.paper_model())
    g, _ = _check(nb, wp, "paper-sized model, cluster")
    assert g.nep_zbl_last_counts()[1] > 20


def test_md_through_a_collision_graph_and_stream_agree(nb, monkeypatch):
    """A 1 keV knock-on in a small crystal: atoms enter the fp64 list and the ZBL range and leave them again while the
    list is rebuilt.  The captured-graph path (both IF nodes taken and not taken) must give the same bits as
    the plain stream launches, and both must follow the oracle."""
    w = wl.bulk_cascade(8, 1000.0, seed=5, n_steps=0, name="pka")
    n_steps = 120
    res = []
    for no_graph in ("0", "1"):
        monkeypatch.setenv("NEPZBL_NO_GRAPH", no_graph)
        g = nb.NepZbl(w.model, w.n)
        pos = torch.from_numpy(w.pos.copy()).cuda(); vel = torch.from_numpy(w.vel.copy()).cuda()
        g.md_init(pos, vel, torch.from_numpy(w.types).cuda(), w.box, w.pbc)
        assert g.nep_zbl_uses_graph() == (no_graph == "0")
        seen_fp64 = seen_zbl = 0
        for _ in range(n_steps):
            g.md_step(w.dt_max, w.max_displacement)
            a, b = g.nep_zbl_last_counts()
            seen_zbl = max(seen_zbl, a); seen_fp64 = max(seen_fp64, b)
        assert seen_fp64 > 0 and seen_zbl > 0
        res.append((pos.cpu().numpy().copy(), vel.cpu().numpy().copy(), g.md_get_counters()[1]))
    assert res[0][0].tobytes() == res[1][0].tobytes() and res[0][1].tobytes() == res[1][1].tobytes()
    assert res[0][2] == res[1][2] and res[0][2] >= 2          # md_init's build and at least one rebuild on the way
    opos, ovel, *_ = oracle.md_run(oracle.Params(w.model), w.pos, w.vel, w.types, w.box, w.pbc, n_steps, w.dt_max,
                                   w.max_displacement)
    L = w.box[[0, 4, 8]][:, None]
    d = res[0][0] - opos
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 2e-5
    # every atom is kicked exactly once per half step, also the ZBL atoms whose second half-kick is k_zbl's: a missed
    # or doubled half-kick of one of them (dt/2 F/m ~ 1e-5 A/fs here) would show up in the velocities
    assert np.abs(res[0][1] - ovel).max() < 2e-6


def test_more_than_64_angular_neighbours(nb):
    """cap_angular up to 128 (two mask words per atom): a cluster dense enough that some atoms have more than 64
    neighbours inside rc_angular + skin = 5 A -- more than any of the paper-shaped cascades here produced (50), but
    what a 100-200 keV core may reach ("cap_angular is capped at 64").  Same tolerances, sets bit-exact."""
    m = wl.synthetic_model(cap_radial=256, cap_angular=128)
    w = wl.free_cluster(n=180, seed=33, radius=5.6, min_sep=1.45, model=m)
    g, _ = _check(nb, w, "dense cluster, cap_angular 128")
    nn, nl = g.neighbor_get(1)
    assert int(nn.max()) > 100, int(nn.max())          # the second mask word is really in use (113 list entries)
    bad, dup, _ = parity.compare_neighbor_sets(nn.cpu().numpy(), nl.cpu().numpy(), w.pos, w.box, w.pbc,
                                               m["rc_angular"] + m["skin"], oracle)
    assert not bad and not dup, (bad[:5], dup[:5])
    # the same capacity on a crystal: the two-word kernels (FFMA network) and the one-word ones (tensor-core network)
    # agree far inside the oracle tolerance
    wc = wl.config1(seed=2, cells=5, n_pairs=1)
    e1, f1, v1 = nb.NepZbl(wc.model, wc.n).compute(wc.pos, wc.types, wc.box, wc.pbc)
    e2, f2, v2 = nb.NepZbl(dict(wc.model, cap_angular=128), wc.n).compute(wc.pos, wc.types, wc.box, wc.pbc)
    assert np.abs(e1 - e2).max() < 3e-6 and np.abs(f1 - f2).max() < 3e-5
