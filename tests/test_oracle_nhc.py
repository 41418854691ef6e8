"""Pins of the oracle's Nose-Hoover-chain thermostat (ref. [32]; DESIGN C-24):
the chain equations of ref. [32] integrated independently (scipy), the conserved quantity, time reversal,
the NVE limit and the target temperature."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_2305_08140_b200 import workloads as wl

KB = 8.617333262e-5
MV2 = 183.84 * 103.6426965  # m in eV fs^2 / A^2


def _small(seed=2, cells=4, T=300.0):
    w = wl.thermal_bulk(cells, seed=seed, temperature=T, sigma_pos=0.03)
    return w, oracle.Params(w.model)


def test_empty_group_is_plain_velocity_verlet():
    w, P = _small()
    a = oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, 6, 1.0, 0.01)
    b = oracle.md_run_nhc(P, w.pos, w.vel, w.types, w.box, w.pbc, 6, 1.0, 0.01,
                          np.zeros(w.n, np.uint8), 300.0, 100.0)
    assert np.array_equal(a[0], b["pos"]) and np.array_equal(a[1], b["vel"]) and np.array_equal(a[2], b["dt"])


def _chain_rhs(t, y, M, nf, kT, Q):
    # y = [ke2, xi_1..M, vxi_1..M]; ref. [32] equations for force-free thermostatted particles
    ke2, vxi = y[0], y[1 + M:]
    d = np.zeros_like(y)
    d[0] = -2.0 * vxi[0] * ke2
    d[1:1 + M] = vxi
    for k in range(M):
        G = (ke2 - nf * kT) / Q[0] if k == 0 else (Q[k - 1] * vxi[k - 1] ** 2 - kT) / Q[k]
        d[1 + M + k] = G - (vxi[k] * vxi[k + 1] if k + 1 < M else 0.0)
    return d


@pytest.mark.parametrize("M", [1, 2, 4])
def test_force_free_particles_follow_the_chain_equations(M):
    # zero network, no ZBL: F = 0; every atom thermostatted: sum m v^2 and the chain obey a closed ODE
    w, _ = _small(T=100.0)
    P = oracle.Params(dict(w.model, w1=np.zeros(50), b1=0.0, zbl_enabled=0))
    T, tau, t_end = 300.0, 20.0, 200.0
    nf, kT = 3.0 * w.n, KB * T
    Q = np.array([nf * kT * tau ** 2] + [kT * tau ** 2] * (M - 1))
    ke2_0 = MV2 * (w.vel ** 2).sum()
    sol = solve_ivp(_chain_rhs, (0.0, t_end), np.concatenate([[ke2_0], np.zeros(2 * M)]),
                    args=(M, nf, kT, Q), rtol=1e-11, atol=1e-14, method="DOP853")
    ref_ke2, ref_xi, ref_vxi = sol.y[0, -1], sol.y[1:1 + M, -1], sol.y[1 + M:, -1]
    errs = []
    for dt in (0.5, 0.25):
        r = oracle.md_run_nhc(P, w.pos, w.vel, w.types, w.box, w.pbc, int(round(t_end / dt)), dt, np.inf,
                              np.ones(w.n, np.uint8), T, tau, chain=M)
        ke2 = MV2 * (r["vel"] ** 2).sum()
        e = max(abs(ke2 / ref_ke2 - 1.0), np.abs(r["xi"] - ref_xi).max() / np.abs(ref_xi).max(),
                np.abs(r["vxi"] - ref_vxi).max() / np.abs(ref_vxi).max())
        errs.append(e)
        # velocities are only rescaled: directions unchanged
        assert np.allclose(r["vel"] / np.linalg.norm(r["vel"]), w.vel / np.linalg.norm(w.vel), atol=1e-12)
    assert errs[0] < 2e-3, errs
    assert 3.0 < errs[0] / errs[1] < 5.0, errs  # second-order splitting
    assert ref_ke2 > 1.2 * ke2_0               # the thermostat is heating the 100 K gas towards 300 K


def test_single_operator_small_step_limit():
    # NHC(delta) -> first order in delta: vxi_1 += G_1 delta, s = 1 - vxi_1 delta
    nf, kT, tau, ke2 = 30.0, 0.02, 50.0, 1.3
    d = 1e-4
    s, xi, vxi = oracle.nhc_half_step(3, nf, kT, tau, d, ke2, np.zeros(3), np.array([2e-3, -1e-3, 5e-4]))
    Q1, Q2 = nf * kT * tau ** 2, kT * tau ** 2
    assert (vxi[0] - 2e-3) / d == pytest.approx((ke2 - nf * kT) / Q1 - 2e-3 * -1e-3, rel=1e-3)
    assert (vxi[1] + 1e-3) / d == pytest.approx((Q1 * 4e-6 - kT) / Q2 - (-1e-3) * 5e-4, rel=1e-3)
    assert (vxi[2] - 5e-4) / d == pytest.approx((Q2 * 1e-6 - kT) / Q2, rel=1e-3)
    assert (1.0 - s) / d == pytest.approx(2e-3, rel=1e-3)
    assert xi / d == pytest.approx([2e-3, -1e-3, 5e-4], rel=1e-3)


def test_conserved_quantity_error_scales_as_dt_squared():
    w, P = _small(T=600.0)
    group = (np.arange(w.n) % 2).astype(np.uint8)
    fl = []
    for dt, n in ((2.0, 20), (1.0, 40), (0.5, 80)):
        r = oracle.md_run_nhc(P, w.pos, w.vel, w.types, w.box, w.pbc, n, dt, np.inf, group, 300.0, 25.0)
        h = r["conserved"]
        fl.append(np.abs(h - h[0]).max())
        # the thermostat does exchange energy: E_kin + E_pot alone is NOT conserved at this level
        e = r["epot"] + r["ekin"]
        assert np.abs(e - e[0]).max() > 20 * fl[-1]
    assert 2.5 < fl[0] / fl[1] < 6.0 and 2.5 < fl[1] / fl[2] < 6.0, fl


def test_time_reversal_with_chain():
    w, P = _small()
    group = (np.arange(w.n) % 3 == 0).astype(np.uint8)
    a = oracle.md_run_nhc(P, w.pos, w.vel, w.types, w.box, w.pbc, 15, 1.0, np.inf, group, 500.0, 30.0)
    b = oracle.md_run_nhc(P, a["pos"], -a["vel"], w.types, w.box, w.pbc, 15, 1.0, np.inf, group, 500.0, 30.0,
                          xi=a["xi"], vxi=-a["vxi"])
    L = w.box[[0, 4, 8]][:, None]
    d = b["pos"] - w.pos
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-9
    assert np.abs(b["vel"] + w.vel).max() < 1e-11 and np.abs(b["vxi"]).max() < 1e-12


def test_group_temperature_goes_to_target():
    w, P = _small(T=100.0)
    group = (np.arange(w.n) % 2).astype(np.uint8)
    r = oracle.md_run_nhc(P, w.pos, w.vel, w.types, w.box, w.pbc, 2500, 1.0, np.inf, group, 300.0, 50.0)
    tg = r["t_group"]
    assert tg[0] == pytest.approx(100.0, rel=0.25)
    assert tg[1000:].mean() == pytest.approx(300.0, rel=0.2)


def test_border_group_generator():
    w = wl.thermal_bulk(10, seed=1)
    g = wl.border_group(w.pos, w.box, w.pbc)
    # 10^3 cells, 3 a0 at each face: inner block is 4^3 cells
    assert g.sum() == w.n - 2 * 4 ** 3
    f = wl.config5(cells=(10, 10, 6))
    gf = wl.border_group(f.pos, f.box, f.pbc)
    assert gf.sum() == f.n - 2 * 4 * 4 * 6  # open z faces are not thermostatted
