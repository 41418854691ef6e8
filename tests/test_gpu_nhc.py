"""GPU tests of the Nose-Hoover-chain thermostat on the border group (ref. [32];
DESIGN C-24): md_set_thermostat + md_step / md_run against the oracle's md_run_nhc."""
import numpy as np
import pytest
import torch

import oracle
from paper_2305_08140_b200 import workloads as wl

pytestmark = pytest.mark.gpu

KB = 8.617333262e-5


@pytest.fixture(scope="module")
def nb():
    from paper_2305_08140_b200 import binding
    assert torch.cuda.is_available()
    return binding


def _md(nb, w, group, T, tau, chain):
    g = nb.NepZbl(w.model, w.n)
    pos = torch.from_numpy(w.pos.copy()).cuda()
    vel = torch.from_numpy(w.vel.copy()).cuda()
    g.md_init(pos, vel, torch.from_numpy(w.types).cuda(), w.box, w.pbc)
    g.md_set_thermostat(torch.from_numpy(group).cuda(), T, tau, chain)
    return g, pos, vel


def _min_image(d, box):
    L = box[[0, 4, 8]][:, None]
    return d - L * np.round(d / L)


@pytest.mark.parametrize("chain", [1, 4])
def test_force_free_chain_matches_oracle_to_rounding(nb, chain):
    # zero network, no ZBL: forces vanish identically on both sides, the whole step is fp64 chain arithmetic
    w = wl.thermal_bulk(6, seed=5, temperature=100.0)
    w.model = dict(w.model, w1=np.zeros(50), b1=0.0, zbl_enabled=0)
    group = (np.arange(w.n) % 3 != 0).astype(np.uint8)
    n = 200
    ref = oracle.md_run_nhc(oracle.Params(w.model), w.pos, w.vel, w.types, w.box, w.pbc, n, 0.5, 0.002,
                            group, 300.0, 20.0, chain=chain)
    g, pos, vel = _md(nb, w, group, 300.0, 20.0, chain)
    tr, _ = g.md_run(n, 0.5, 0.002, want_trace=True)
    xi, vxi, tg, extra = g.md_get_thermostat()
    assert np.allclose(tr, ref["dt"], rtol=1e-12, atol=0)
    assert tr.min() < 0.5                                      # the adaptive step was active
    assert np.abs(vel.cpu().numpy() - ref["vel"]).max() < 1e-13 * np.abs(ref["vel"]).max() * n
    assert np.abs(_min_image(pos.cpu().numpy() - ref["pos"], w.box)).max() < 1e-10
    assert np.allclose(xi, ref["xi"], rtol=1e-10, atol=1e-14) and np.allclose(vxi, ref["vxi"], rtol=1e-10, atol=1e-16)
    assert tg == pytest.approx(ref["t_group"][-1], rel=1e-10)
    ep, ek = g.md_energies()
    assert ep + ek + extra == pytest.approx(ref["conserved"][-1], rel=1e-10)
    # untouched atoms kept their velocities exactly
    assert np.array_equal(vel.cpu().numpy()[:, group == 0], w.vel[:, group == 0])


def test_trajectory_with_forces_follows_oracle(nb):
    w = wl.thermal_bulk(6, seed=6, temperature=150.0, sigma_pos=0.03)
    group = wl.border_group(w.pos, w.box, w.pbc, thickness=wl.A0_CONFIG)
    assert 0 < group.sum() < w.n
    n = 40
    ref = oracle.md_run_nhc(oracle.Params(w.model), w.pos, w.vel, w.types, w.box, w.pbc, n, 1.0, np.inf,
                            group, 300.0, 25.0, chain=4)
    g, pos, vel = _md(nb, w, group, 300.0, 25.0, 4)
    for _ in range(n):
        g.md_step(1.0, float("inf"))
    xi, vxi, tg, extra = g.md_get_thermostat()
    d = _min_image(pos.cpu().numpy() - ref["pos"], w.box)
    print("NHC: max|dx| =", np.abs(d).max(), "max|dv| =", np.abs(vel.cpu().numpy() - ref["vel"]).max(),
          "xi", xi, ref["xi"])
    assert np.abs(d).max() < 5e-6 and np.abs(vel.cpu().numpy() - ref["vel"]).max() < 5e-7
    assert np.allclose(xi, ref["xi"], rtol=1e-4, atol=1e-9) and np.allclose(vxi, ref["vxi"], rtol=1e-4, atol=1e-10)
    assert tg == pytest.approx(ref["t_group"][-1], rel=1e-4)
    ep, ek = g.md_energies()
    assert ep + ek + extra == pytest.approx(ref["conserved"][-1], abs=2e-5 * w.n)
    assert abs(ref["vxi"][0]) > 1e-4   # the chain did act on this run


def test_md_run_graph_equals_md_step_and_switch_off(nb):
    w = wl.thermal_bulk(6, seed=7, sigma_pos=0.03)
    group = wl.border_group(w.pos, w.box, w.pbc, thickness=wl.A0_CONFIG)
    g1, p1, v1 = _md(nb, w, group, 300.0, 50.0, 3)
    g2, p2, v2 = _md(nb, w, group, 300.0, 50.0, 3)
    g1.md_run(25, 1.0, 0.01)
    for _ in range(25):
        g2.md_step(1.0, 0.01)
    assert torch.equal(p1, p2) and torch.equal(v1, v2)          # bitwise: deterministic reductions
    assert np.array_equal(g1.md_get_thermostat()[1], g2.md_get_thermostat()[1])
    # switched off -> plain NVE again, as a handle that never had a thermostat (its list is newer, so the
    # fp32 summation order differs: equal to rounding, not bitwise)
    g3 = nb.NepZbl(w.model, w.n)
    p3, v3 = p1.clone(), v1.clone()
    g3.md_init(p3, v3, torch.from_numpy(w.types).cuda(), w.box, w.pbc)
    g1.md_set_thermostat(None, 300.0, 50.0, 3)
    g1.md_run(5, 1.0, 0.01)
    g3.md_run(5, 1.0, 0.01)
    assert (p1 - p3).abs().max().item() < 1e-8 and (v1 - v3).abs().max().item() < 1e-9


def test_graph_path_is_active_and_equals_stream_launches_with_thermostat(nb, monkeypatch):
    """The captured-graph step (what bench.py and every DESIGN.md number measure) against the same kernels as plain
    stream launches (NEPZBL_NO_GRAPH=1), bit for bit, on a thermostatted cascade cell where both IF nodes (list
    rebuild, ZBL) and the fp64 pass fire."""
    w = wl.bulk_cascade(8, 800.0, seed=15, n_steps=0, name="nhc_graph")
    group = wl.border_group(w.pos, w.box, w.pbc, thickness=wl.A0_CONFIG)
    out = []
    for no_graph in ("0", "1"):
        monkeypatch.setenv("NEPZBL_NO_GRAPH", no_graph)
        g, pos, vel = _md(nb, w, group, 300.0, 50.0, 4)
        assert g.nep_zbl_uses_graph() == (no_graph == "0")
        g.md_run(150, 1.0, 0.015)
        steps, rebuilds, _ = g.md_get_counters()
        out.append((pos.cpu().numpy().copy(), vel.cpu().numpy().copy(), g.md_get_thermostat()[1].copy(), rebuilds))
    assert out[0][3] == out[1][3] and out[0][3] >= 2
    for a, b in zip(out[0][:3], out[1][:3]):
        assert a.tobytes() == b.tobytes()


def test_border_layer_of_a_cascade_cell(nb):
    # 24^3 cells (27 648 atoms), 3 a0 border layer, 2 keV PKA at the centre, adaptive step: the
    # group temperature reported by the library is the group's, and the conserved quantity of ref. [32] holds
    w = wl.bulk_cascade(24, 2.0e3, seed=8, n_steps=400, name="nhc_cascade")
    group = wl.border_group(w.pos, w.box, w.pbc)
    assert group.sum() == w.n - 2 * 18 ** 3
    g, pos, vel = _md(nb, w, group, 300.0, 100.0, 4)
    e0 = sum(g.md_energies())
    tr, _ = g.md_run(400, 1.0, 0.015, want_trace=True)
    xi, vxi, tg, extra = g.md_get_thermostat()
    ep, ek = g.md_energies()
    v = vel.cpu().numpy()
    tg_host = wl.W_MASS * wl.AMU_A2_FS2_TO_EV * (v[:, group == 1] ** 2).sum() / (3 * group.sum() * KB)
    assert tg == pytest.approx(tg_host, rel=1e-12)
    assert tr.max() <= 1.0 and tr.min() < 0.2
    assert abs(ep + ek + extra - e0) / w.n < 2e-4 and np.isfinite(xi).all()


def test_border_layer_is_held_at_the_target_temperature(nb):
    # a perfect lattice given 300 K velocities settles at ~150 K kinetic temperature (equipartition); with
    # the border layer thermostatted at 300 K the layer is driven to 300 K, without it it is not
    w = wl.thermal_bulk(16, seed=9)
    group = wl.border_group(w.pos, w.box, w.pbc)
    g, pos, vel = _md(nb, w, group, 300.0, 50.0, 4)
    e0 = sum(g.md_energies())
    g.md_run(1500, 1.0, float("inf"))
    tgs = []
    for _ in range(50):
        g.md_run(10, 1.0, float("inf"))
        tgs.append(g.md_get_thermostat()[2])
    xi, vxi, tg, extra = g.md_get_thermostat()
    ep, ek = g.md_energies()
    print("NHC border layer: <T_group> =", np.mean(tgs), " dH/N =", (ep + ek + extra - e0) / w.n)
    assert np.mean(tgs) == pytest.approx(300.0, rel=0.1)
    assert abs(ep + ek + extra - e0) / w.n < 5e-4
    g.md_set_thermostat(None, 300.0, 50.0, 4)
    w2 = wl.thermal_bulk(16, seed=9)
    g2 = nb.NepZbl(w2.model, w2.n)
    p2 = torch.from_numpy(w2.pos.copy()).cuda(); v2 = torch.from_numpy(w2.vel.copy()).cuda()
    g2.md_init(p2, v2, torch.from_numpy(w2.types).cuda(), w2.box, w2.pbc)
    g2.md_run(1500, 1.0, float("inf"))
    vv = v2.cpu().numpy()
    t_nve = wl.W_MASS * wl.AMU_A2_FS2_TO_EV * (vv[:, group == 1] ** 2).sum() / (3 * group.sum() * KB)
    assert t_nve < 200.0


def test_resume_from_saved_state(nb):
    # checkpoint / resume: positions, velocities and the chain state are all a run needs
    w = wl.thermal_bulk(6, seed=10, sigma_pos=0.03)
    group = wl.border_group(w.pos, w.box, w.pbc, thickness=wl.A0_CONFIG)
    g1, p1, v1 = _md(nb, w, group, 300.0, 40.0, 4)
    g1.md_run(15, 1.0, 0.01)
    xi, vxi, _, _ = g1.md_get_thermostat()
    w2 = wl.thermal_bulk(6, seed=10, sigma_pos=0.03)
    w2.pos, w2.vel = p1.cpu().numpy().copy(), v1.cpu().numpy().copy()
    g2, p2, v2 = _md(nb, w2, group, 300.0, 40.0, 4)
    g2.md_set_thermostat_state(xi, vxi)
    g1.md_run(15, 1.0, 0.01)
    g2.md_run(15, 1.0, 0.01)
    # the resumed handle rebuilt its list (other fp32 summation order): equal to rounding
    assert (p1 - p2).abs().max().item() < 1e-8 and (v1 - v2).abs().max().item() < 1e-9
    assert np.allclose(g1.md_get_thermostat()[1], g2.md_get_thermostat()[1], rtol=1e-7, atol=1e-12)


def test_cascade_example_runs(nb, capsys):
    # the packaged protocol example (PKA + adaptive dt + border thermostat + Wigner-Seitz counts) on a small cell
    from paper_2305_08140_b200 import cascade_example
    assert cascade_example.main(["--cells", "12", "--energy-kev", "0.5", "--steps", "120", "--every", "60"]) == 0
    out = capsys.readouterr().out
    assert "step    120" in out and "atom-steps/s" in out
