"""Pins of the oracle's integrator (adaptive step P:77): things any correct
velocity-Verlet must satisfy -- time reversal, energy error ~ dt^2, the displacement cap."""
import numpy as np
import pytest

import oracle
from paper_2305_08140_b200 import workloads as wl


def _small(seed=2, cells=4, T=300.0):
    w = wl.thermal_bulk(cells, seed=seed, temperature=T, sigma_pos=0.03)
    return w, oracle.Params(w.model)


def test_free_flight_without_forces():
    # zero network + no ZBL: F = 0, so x(t) = x0 + v t exactly and dt = dt_max
    w, _ = _small()
    m = dict(w.model, w1=np.zeros(50), b1=0.0, zbl_enabled=0)
    P = oracle.Params(m)
    pos, vel, dt, ep, ek = oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, 7, 0.5, np.inf)
    L = w.box[[0, 4, 8]][:, None]
    assert np.all(dt == 0.5)
    d = pos - np.mod(w.pos + 3.5 * w.vel, L)
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-12
    assert np.array_equal(vel, w.vel) and np.all(ep == 0) and np.ptp(ek) < 1e-15 * ek[0] + 1e-18
    # kinetic energy: sum 1/2 m v^2 in eV (unit constant 103.6426965)
    assert ek[0] == pytest.approx(0.5 * 183.84 * 103.6426965 * (w.vel ** 2).sum(), rel=1e-14)
    # equipartition sanity of the generator: <Ek> = 3/2 kB T per atom within sampling noise
    assert ek[0] / w.n == pytest.approx(1.5 * 8.617333262e-5 * 300.0, rel=0.15)


def test_time_reversal():
    w, P = _small()
    n = 20
    pos1, vel1, dt1, _, _ = oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, n, 1.0, np.inf)
    pos2, vel2, dt2, _, _ = oracle.md_run(P, pos1, -vel1, w.types, w.box, w.pbc, n, 1.0, np.inf)
    L = w.box[[0, 4, 8]][:, None]
    d = pos2 - w.pos
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-9
    assert np.abs(vel2 + w.vel).max() < 1e-11


def test_energy_error_scales_as_dt_squared():
    w, P = _small(T=600.0)
    errs = []
    for dt, n in ((2.0, 20), (1.0, 40), (0.5, 80)):
        _, _, _, ep, ek = oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, n, dt, np.inf)
        e = ep + ek
        errs.append(np.abs(e - e[0]).max())
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.35)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.35)
    assert errs[2] / w.n < 1e-4


def test_adaptive_time_step_caps_the_displacement():
    # a 1 keV knock-on in a small cell: dt = max_disp / v_max < dt_max, and no atom moves more than
    # max_disp (1 + O(dt^2)) in a step; once everything is slow dt returns to dt_max (C-11)
    w, P = _small(cells=4)
    v = w.vel.copy()
    vp = wl.pka_speed(1000.0, wl.W_MASS)
    v[:, 5] = vp * np.array([1.0, 3.0, 5.0]) / np.sqrt(35.0)
    pos, vel = w.pos, v
    L = w.box[[0, 4, 8]][:, None]
    for _ in range(5):
        vmax = np.sqrt((vel ** 2).sum(axis=0)).max()
        p2, v2, dt, _, _ = oracle.md_run(P, pos, vel, w.types, w.box, w.pbc, 1, 1.0, 0.015)
        assert dt[0] == pytest.approx(min(1.0, 0.015 / vmax), rel=1e-14)
        d = p2 - pos
        d -= L * np.round(d / L)
        assert np.sqrt((d ** 2).sum(axis=0)).max() <= 0.015 * (1 + 1e-3)
        pos, vel = p2, v2
    assert dt[0] < 0.05
    slow = np.zeros_like(w.vel)
    _, _, dt, _, _ = oracle.md_run(P, w.pos, slow, w.types, w.box, w.pbc, 1, 1.0, 0.015)
    assert dt[0] == 1.0                            # v_max = 0 -> dt_max


def test_pka_speed_values():
    # 10 keV -> 1.02453 A/fs, 100 keV -> 3.23986 A/fs for W
    assert wl.pka_speed(1.0e4, wl.W_MASS) == pytest.approx(1.02453, rel=1e-5)
    assert wl.pka_speed(1.0e5, wl.W_MASS) == pytest.approx(3.23986, rel=1e-5)


def test_paper_sized_model_keeps_the_crystal():
    # SURVEY 8(f) NEXT-2 input recipe: the seeded paper-sized potential (workloads.paper_model) must hold bcc W
    # at 300 K, otherwise the "paper" workload would not have the paper's neighbour structure (58 / 14)
    w = wl.paper_bulk(4, seed=12)
    P = oracle.Params(w.model)
    assert P.D == 60 and w.model["n_neurons"] == 100
    pos, vel, dt, ep, ek = oracle.md_run(P, w.pos, w.vel, w.types, w.box, w.pbc, 300, 1.0, 0.01)
    L = w.box[[0, 4, 8]][:, None]
    d = pos - w.pos
    d -= L * np.round(d / L)
    e = ep + ek
    assert np.abs(d).max() < 0.5 and np.abs(e - e[0]).max() / w.n < 2e-4
    nn, _ = oracle.neighbors(pos, w.box, w.pbc, 6.0)
    na, _ = oracle.neighbors(pos, w.box, w.pbc, 4.0)
    assert np.all(nn == 58) and np.all(na == 14)
