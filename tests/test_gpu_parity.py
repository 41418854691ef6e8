"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element,
on the same seeded inputs.  Tolerances: BASELINE.json north_star (see tests/parity.py)."""
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
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return binding


def _run(nb, w, virial=True, model=None, n_cap=None):
    m = model or w.model
    g = nb.NepZbl(m, n_cap or w.n)
    e, f, v = g.compute(w.pos, w.types, w.box, w.pbc, virial=virial)
    return g, e, f, v


def _assert_ok(r):
    for k, v in r.items():
        assert v <= 1.0, (k, v)


# ------------------------------------------------------------------ config 1: full parity

def test_config1_energy_force_virial(nb):
    w = wl.config1()
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)
    g, e, f, v = _run(nb, w)
    _assert_ok(parity.compare(e, f, v, ref, label="config1"))
    # the pushed pairs carry ZBL energies of tens of eV and are inside the same tolerance
    zi = [a for p in w.info["pairs"] for a in p]
    assert ref.energy[zi].max() > 1.0
    _assert_ok(parity.compare(e, f, v, ref, idx=np.array(zi), label="config1 ZBL atoms"))
    # totals
    assert abs(e.sum() - ref.energy.sum()) < 1e-5 * np.sqrt(w.n) * 3
    assert np.abs(f.sum(axis=1)).max() < 2e-3          # zero net force up to fp32 rounding


def test_config1_descriptors(nb):
    w = wl.config1()
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, want_q=True,
                         want_force=False, want_virial=False)
    g, e, f, v = _run(nb, w)
    q = g.nep_zbl_get_descriptors().cpu().numpy()
    scale = np.asarray(w.model["q_scaler"])
    err = np.abs(q - ref.q) * scale          # in units of the network input
    print("descriptor err (scaled) per block:", [float(err[:, s].max()) for s in
          (slice(0, 5), slice(5, 10), slice(10, 15), slice(15, 20), slice(20, 25), slice(25, 30))])
    # fp32 sums: absolute 2e-5 in network-input units plus 3e-6 relative (large 4-body values next
    # to the pushed pairs carry a proportionally larger rounding error)
    assert (err / (2e-5 + 3e-6 * np.abs(ref.q * scale))).max() < 1.0


def test_config1_neighbor_sets(nb):
    w = wl.config1()
    for skin in (1.0, 0.0):
        m = dict(w.model, skin=skin)
        g = nb.NepZbl(m, w.n)
        pos = torch.from_numpy(w.pos).cuda(); types = torch.from_numpy(w.types).cuda()
        g.neighbor_build(pos, types, w.box, w.pbc)
        for which, rc in ((0, 6.0 + skin), (1, 4.0 + skin)):
            nn, nl = g.neighbor_get(which)
            bad, dup, amb = parity.compare_neighbor_sets(nn.cpu().numpy(), nl.cpu().numpy(), w.pos, w.box,
                                                         w.pbc, rc, oracle)
            assert not bad and not dup, (skin, which, bad[:5], dup[:5])


def test_config1_block_isolated(nb):
    """parity with all but one descriptor block's W0 columns zeroed."""
    w = wl.config1()
    blocks = dict(radial=slice(0, 5), l1=slice(5, 10), l2=slice(10, 15), l3=slice(15, 20),
                  l4=slice(20, 25), fourbody=slice(25, 30))
    for name, sl in blocks.items():
        w0 = np.zeros_like(w.model["w0"]); w0[:, sl] = w.model["w0"][:, sl]
        m = dict(w.model, w0=w0)
        ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
        g, e, f, v = _run(nb, w, model=m)
        _assert_ok(parity.compare(e, f, v, ref, label=f"block {name}"))


def test_bitwise_determinism(nb):
    w = wl.config1(seed=3)
    outs = []
    for _ in range(3):
        g, e, f, v = _run(nb, w)
        outs.append((e.copy(), f.copy(), v.copy()))
    for o in outs[1:]:
        for a, b in zip(outs[0], o):
            assert a.tobytes() == b.tobytes()
    # a shuffled atom order changes the in-cell order (ascending caller index), hence the fp32
    # summation order: same values to rounding, not the same bits
    perm = wl.rng(3, 20).permutation(w.n)
    g = nb.NepZbl(w.model, w.n)
    e2, f2, v2 = g.compute(w.pos[:, perm], w.types[perm], w.box, w.pbc)
    assert np.abs(e2 - outs[0][0][perm]).max() < 1e-5
    assert np.abs(f2 - outs[0][1][:, perm]).max() < 1e-3


def test_no_4body_shape_and_no_zbl(nb):
    w = wl.config1(seed=4, cells=6)
    m = wl.synthetic_model(has_4body=0)
    m["zbl_enabled"] = 0
    ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
    g, e, f, v = _run(nb, w, model=m)
    _assert_ok(parity.compare(e, f, v, ref, label="no 4-body, no ZBL"))


def test_paper_eq3_screening_function(nb):
    w = wl.config1(seed=5, cells=6)
    m = wl.synthetic_model(zbl="paper")
    ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
    g, e, f, v = _run(nb, w, model=m)
    _assert_ok(parity.compare(e, f, v, ref, label="Eq.3 phi"))


# ------------------------------------------------------------------ geometry edge cases

def test_translation_and_unwrapped_positions(nb):
    w = wl.config1(seed=6, cells=6)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)
    shift = np.array([[3.3], [-47.9], [125.1]])
    g = nb.NepZbl(w.model, w.n)
    e, f, v = g.compute(w.pos + shift, w.types, w.box, w.pbc)
    _assert_ok(parity.compare(e, f, v, ref, label="shifted/unwrapped"))


def test_minimum_box_two_cells_per_axis(nb):
    # periodic edge 15.825 A: exactly 2 cells of >= 7 A per axis (the stencil must not double count)
    w = wl.config1(seed=7, cells=5, n_pairs=2)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, use_cell=False)
    g, e, f, v = _run(nb, w)
    _assert_ok(parity.compare(e, f, v, ref, label="2 cells/axis"))
    g2 = nb.NepZbl(w.model, w.n)
    pos = torch.from_numpy(w.pos).cuda()
    g2.neighbor_build(pos, None, w.box, w.pbc)
    nn, nl = g2.neighbor_get(0)
    bad, dup, _ = parity.compare_neighbor_sets(nn.cpu().numpy(), nl.cpu().numpy(), w.pos, w.box, w.pbc, 7.0, oracle)
    assert not bad and not dup


def test_open_boundaries_foil_and_cluster(nb):
    # small foil: periodic x,y, open z with vacuum; atoms outside the nominal box in z
    wf = wl.config5(seed=5, cells=(6, 6, 4), vacuum=20.0)
    wf.pos = wf.pos + wl.rng(5, 21).standard_normal(wf.pos.shape) * 0.05
    wf.pos[2, :7] -= 30.0                           # a few atoms sputtered below the box
    ref = oracle.compute(oracle.Params(wf.model), wf.pos, wf.types, wf.box, wf.pbc, use_cell=False)
    g, e, f, v = _run(nb, wf)
    _assert_ok(parity.compare(e, f, v, ref, label="foil"))
    nn, nl = g.neighbor_get(0)
    bad, dup, _ = parity.compare_neighbor_sets(nn.cpu().numpy(), nl.cpu().numpy(), wf.pos, wf.box, wf.pbc, 7.0, oracle)
    assert not bad and not dup
    # free bcc nano-particle (all axes open) with two ZBL pairs
    wc = wl.config1(seed=8, cells=4, n_pairs=2)
    wc.pos = wc.pos + 30.0
    wc.box = np.diag([100.0, 100.0, 100.0]).ravel()
    wc.pbc = np.zeros(3, dtype=np.int32)
    ref = oracle.compute(oracle.Params(wc.model), wc.pos, wc.types, wc.box, wc.pbc, use_cell=False)
    g, e, f, v = _run(nb, wc)
    _assert_ok(parity.compare(e, f, v, ref, label="free particle"))
    # a dense RANDOM cluster (pairs down to 1.7 A everywhere): disordered sites go through the fp64 pass of
    # csrc/site_fp64.cuh and meet the same tolerance (more cases in tests/test_gpu_disordered.py)
    wr = wl.free_cluster(n=60, seed=8, radius=7.0, min_sep=1.7)
    ref = oracle.compute(oracle.Params(wr.model), wr.pos, wr.types, wr.box, wr.pbc, use_cell=False)
    g, e, f, v = _run(nb, wr)
    _assert_ok(parity.compare(e, f, v, ref, label="random cluster"))


def test_dimer_closed_form_zbl(nb):
    # two atoms, zero network: E_i = 1/2 U_ZBL(r), F = -dU/dr (Eq. 1-4)
    m = wl.synthetic_model()
    m["w1"] = np.zeros_like(m["w1"]); m["b1"] = 0.0
    P = oracle.Params(m)
    for r in (0.6, 1.0, 1.37, 1.95, 2.5):
        pos = np.array([[10.0, 10.0 + r], [10.0, 10.0], [10.0, 10.0]])
        g = nb.NepZbl(m, 2)
        e, f, v = g.compute(pos, np.zeros(2, np.int32), np.diag([40.0, 40, 40]).ravel(), [0, 0, 0])
        u, du = oracle.zbl_pair(P, r)
        assert e == pytest.approx([0.5 * u, 0.5 * u], rel=1e-12, abs=1e-12)
        assert f[0] == pytest.approx([du, -du], rel=2e-7, abs=1e-6)
        assert v[0].sum() == pytest.approx(-r * du, rel=2e-7, abs=1e-6)


def test_single_atom_and_empty(nb):
    m = wl.synthetic_model()
    g = nb.NepZbl(m, 4)
    pos = np.array([[1.0], [2.0], [3.0]])
    e, f, v = g.compute(pos, np.zeros(1, np.int32), np.diag([30.0, 30, 30]).ravel(), [1, 1, 1])
    ref = oracle.compute(oracle.Params(m), pos, None, np.diag([30.0, 30, 30]).ravel(), [1, 1, 1])
    assert e == pytest.approx(ref.energy, abs=1e-6) and np.all(f == 0)
    e, f, v = g.compute(np.zeros((3, 0)), np.zeros(0, np.int32), np.diag([30.0, 30, 30]).ravel(), [1, 1, 1])
    assert e.size == 0


def test_error_codes(nb):
    w = wl.config1(seed=9, cells=5, n_pairs=0)
    g = nb.NepZbl(w.model, w.n)
    with pytest.raises(nb.NepZblError) as ei:                      # non-orthogonal box with an open axis
        box = w.box.copy(); box[1] = 0.5
        g.compute(w.pos, w.types, box, [1, 1, 0])
    assert ei.value.code == -2
    with pytest.raises(nb.NepZblError) as ei:                      # periodic edge < 2 (rc+skin)
        g.compute(w.pos, w.types, np.diag([13.0, 40, 40]).ravel(), w.pbc)
    assert ei.value.code == -3
    with pytest.raises(nb.NepZblError) as ei:                      # NaN position
        p = w.pos.copy(); p[1, 3] = np.nan
        g.compute(p, w.types, w.box, w.pbc)
    assert ei.value.code == -5
    with pytest.raises(nb.NepZblError) as ei:                      # more atoms than the workspace holds
        w2 = wl.config1(seed=9, cells=6, n_pairs=0)
        g.compute(w2.pos, w2.types, w2.box, w2.pbc)
    assert ei.value.code == -8
    gs = nb.NepZbl(dict(w.model, cap_radial=64), w.n)              # 88 neighbours do not fit 64 slots
    with pytest.raises(nb.NepZblError) as ei:
        gs.compute(w.pos, w.types, w.box, w.pbc)
    import re
    assert ei.value.code == -4
    assert int(re.search(r"needs (\d+) radial", str(ei.value)).group(1)) >= 88   # the atom and its count are reported
    g.compute(w.pos, w.types, w.box, w.pbc)                        # the handle is still usable


def test_list_reuse_within_skin_and_rebuild_beyond(nb):
    w = wl.config1(seed=10, cells=6)
    g = nb.NepZbl(w.model, w.n)
    g.compute(w.pos, w.types, w.box, w.pbc)
    rng = wl.rng(10, 22)
    # small move (< skin/2): list reused, results must still match the oracle at the new positions
    p2 = w.pos + rng.uniform(-0.2, 0.2, size=w.pos.shape)
    l0 = g.nep_zbl_launch_count()
    e, f, v = g.compute(p2, w.types, w.box, w.pbc)
    ref = oracle.compute(oracle.Params(w.model), p2, w.types, w.box, w.pbc)
    _assert_ok(parity.compare(e, f, v, ref, label="reuse list"))
    # big move of one atom (> skin/2): must rebuild
    p3 = p2.copy(); p3[:, 11] += np.array([0.9, -0.8, 0.7])
    e, f, v = g.compute(p3, w.types, w.box, w.pbc)
    ref = oracle.compute(oracle.Params(w.model), p3, w.types, w.box, w.pbc)
    _assert_ok(parity.compare(e, f, v, ref, label="rebuilt list"))


# ------------------------------------------------------------------ at bench size, sampled (north_star)

def test_config2_sampled_parity_at_full_size(nb):
    w = wl.config2()
    w.pos = np.mod(w.pos + wl.rng(2, 23).standard_normal(w.pos.shape) * 0.05, w.box[[0, 4, 8]][:, None])
    g, e, f, v = _run(nb, w)
    sel = np.sort(wl.rng(2, 24).choice(w.n, size=1024, replace=False)).astype(np.int32)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc, sel=sel)
    _assert_ok(parity.compare(e, f, v, ref, idx=sel, label="config2 sample"))
    assert np.abs(f.sum(axis=1)).max() < 0.05


def test_neighbor_sets_with_a_large_capacity(nb):
    # cap_radial above k_nbr's per-thread buffer (192) takes the two-walk path of the list build
    w = wl.config1(seed=12, cells=6)
    m = dict(w.model, cap_radial=256)
    g = nb.NepZbl(m, w.n)
    pos = torch.from_numpy(w.pos).cuda(); types = torch.from_numpy(w.types).cuda()
    g.neighbor_build(pos, types, w.box, w.pbc)
    for which, rc in ((0, 7.0), (1, 5.0)):
        nn, nl = g.neighbor_get(which)
        bad, dup, _ = parity.compare_neighbor_sets(nn.cpu().numpy(), nl.cpu().numpy(), w.pos, w.box, w.pbc, rc, oracle)
        assert not bad and not dup
    ref = oracle.compute(oracle.Params(m), w.pos, w.types, w.box, w.pbc)
    e, f, v = g.compute(w.pos, w.types, w.box, w.pbc)
    _assert_ok(parity.compare(e, f, v, ref, label="cap_radial 256"))


@pytest.mark.parametrize("mode,code", [("ffma", 0), ("mma", 1), ("tcsync", 2), ("tc", 3)])
def test_every_network_path_meets_the_tolerances(nb, monkeypatch, mode, code):
    """The network layer exists in four forms (include/nepzbl.h: nep_zbl_network_mode; profiles/r2_nn_tensor.md); the
    default is the pipelined tcgen05 kernel, the others stay selectable for the measurement.  Each against the oracle,
    energy / force / virial and a short MD run."""
    monkeypatch.setenv("NEPZBL_NN", mode)
    w = wl.config1(seed=4, cells=6, n_pairs=3)
    ref = oracle.compute(oracle.Params(w.model), w.pos, w.types, w.box, w.pbc)
    g = nb.NepZbl(w.model, w.n)
    assert g.nep_zbl_network_mode() == code
    r = parity.compare(*g.compute(w.pos, w.types, w.box, w.pbc), ref, label=f"network path {mode}")
    assert max(r.values()) <= 1.0, (mode, r)
    # ragged tile counts: 1 atom, 33 atoms, 129 atoms of a cluster (partly filled 32- / 128-atom tiles)
    for n_at in (33, 129):
        c = wl.free_cluster(n=n_at, seed=40 + n_at, radius=3.0 * n_at ** (1.0 / 3.0), min_sep=2.2)
        refc = oracle.compute(oracle.Params(c.model), c.pos, c.types, c.box, c.pbc, use_cell=False)
        rc = parity.compare(*nb.NepZbl(c.model, c.n).compute(c.pos, c.types, c.box, c.pbc), refc, label=f"{mode}, {n_at} atoms")
        assert max(rc.values()) <= 1.0, (mode, n_at, rc)


def test_default_network_path_is_the_tensor_core_pipeline(nb, monkeypatch):
    monkeypatch.delenv("NEPZBL_NN", raising=False)
    w = wl.config1(seed=4, cells=5, n_pairs=1)
    assert nb.NepZbl(w.model, w.n).nep_zbl_network_mode() == 3
    assert nb.NepZbl(dict(w.model, cap_angular=128), w.n).nep_zbl_network_mode() == 0     # two mask words: FFMA kernel
