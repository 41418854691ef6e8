"""Pins of the oracle's ZBL pair term against what the paper and the mathematics fix.

Eq. 2-4, Tersoff switch 1.0 -> 2.0 A, Eq. 1 factor 1/2.
None of these tests calls the CUDA path.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2305_08140_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
K_CODATA = 14.3996454784  # e^2/(4 pi eps0) in eV*A


def _params(**over):
    m = wl.synthetic_model()
    m.update(over)
    return oracle.Params(m)


def test_coulomb_limit_textbook():
    # phi == 1, no switch inside r_inner: U = K Z_i Z_j / r.  Two unit charges at 1 A: 14.3996 eV (textbook).
    P = _params(zbl_c=[1.0], zbl_d=[0.0], atomic_number=[1.0], zbl_r_inner=5.0, zbl_r_outer=6.0,
                coulomb_k=K_CODATA)
    u, du = oracle.zbl_pair(P, 1.0)
    assert u == pytest.approx(14.3996454784, rel=1e-14)
    assert du == pytest.approx(-14.3996454784, rel=1e-14)
    u2, _ = oracle.zbl_pair(P, 2.0)
    assert u2 == pytest.approx(u / 2, rel=1e-14)
    P74 = _params(zbl_c=[1.0], zbl_d=[0.0], zbl_r_inner=5.0, zbl_r_outer=6.0, coulomb_k=K_CODATA)
    assert oracle.zbl_pair(P74, 1.0)[0] == pytest.approx(74 * 74 * K_CODATA, rel=1e-14)


def test_screening_length_eq4():
    vals = dict(l.split() for l in open(os.path.join(GOLD, "zbl_constants.txt")) if not l.startswith("#"))
    P = _params()
    a = oracle.zbl_screening_length(P)
    assert a == pytest.approx(float(vals["a_angstrom"]), rel=2e-9)
    assert 0.46848 / (2 * a) == pytest.approx(float(vals["Z_pow_0.23"]), rel=2e-9)


@pytest.mark.parametrize("name,zbl", [("universal", wl.ZBL_UNIVERSAL), ("paper_eq3", wl.ZBL_PAPER_W)])
def test_phi_at_zero_is_sum_of_coefficients(name, zbl):
    # U r / (K Z^2) -> phi(0) = sum c_k  (=1 universal; 1.00154 for Eq. 3 as printed, SURVEY C-9)
    P = _params(**zbl)
    r = 1e-12
    u, _ = oracle.zbl_pair(P, r)
    phi0 = u * r / (P.c.coulomb_k * 74 * 74)
    assert phi0 == pytest.approx(sum(zbl["zbl_c"]), rel=1e-9)
    if name == "universal":
        assert phi0 == pytest.approx(1.0, abs=1e-9)
    else:
        assert phi0 == pytest.approx(1.00154, abs=1e-9)


@pytest.mark.parametrize("zbl", [wl.ZBL_UNIVERSAL, wl.ZBL_PAPER_W])
def test_against_high_precision_closed_form(zbl):
    # independent 40-digit evaluation of Eq. 2-4 with the printed coefficients
    mp.mp.dps = 40
    P = _params(**zbl)
    a = mp.mpf("0.46848") / (2 * mp.mpf(74) ** mp.mpf("0.23"))
    for r in [0.05, 0.3, 0.5, 0.99, 1.0, 1.0001, 1.25, 1.5, 1.75, 1.9999]:
        x = mp.mpf(r) / a
        phi = sum(mp.mpf(repr(c)) * mp.e ** (-mp.mpf(repr(d)) * x) for c, d in zip(zbl["zbl_c"], zbl["zbl_d"]))
        fc = 1 if r <= 1.0 else (mp.mpf(1) / 2 + mp.cos(mp.pi * (mp.mpf(r) - 1) / 1) / 2)
        ref = mp.mpf(repr(P.c.coulomb_k)) * 74 * 74 / mp.mpf(r) * phi * fc
        u, _ = oracle.zbl_pair(P, r)
        assert u == pytest.approx(float(ref), rel=1e-12, abs=1e-12)


def test_survey_dimer_values():
    rows = [l.split() for l in open(os.path.join(GOLD, "zbl_dimer_survey.txt")) if not l.startswith("#")]
    for name, r, u_ref in rows:
        zbl = wl.ZBL_UNIVERSAL if name == "universal" else wl.ZBL_PAPER_W
        P = _params(coulomb_k=K_CODATA, **zbl)
        u, _ = oracle.zbl_pair(P, float(r))
        assert u == pytest.approx(float(u_ref), rel=2e-10, abs=1e-12)


def test_switch_limits_and_smoothness():
    P = _params()
    Pn = _params(zbl_r_inner=50.0, zbl_r_outer=60.0)  # switch == 1 everywhere tested
    for r in (0.2, 0.7, 1.0):  # below r_inner: pure Coulomb*phi
        assert oracle.zbl_pair(P, r) == pytest.approx(oracle.zbl_pair(Pn, r), rel=1e-15)
    # midpoint of the cosine switch: f_c = 1/2
    assert oracle.zbl_pair(P, 1.5)[0] == pytest.approx(0.5 * oracle.zbl_pair(Pn, 1.5)[0], rel=1e-14)
    for r in (2.0, 2.0000001, 3.0, 5.9):  # zero at and beyond r_outer
        assert oracle.zbl_pair(P, r) == (0.0, 0.0)
    # C^1 at both ends: U continuous, dU/dr continuous
    e = 1e-9
    for r0 in (1.0, 2.0):
        ul, dl = oracle.zbl_pair(P, r0 - e)
        ur, dr = oracle.zbl_pair(P, r0 + e)
        assert ul == pytest.approx(ur, abs=1e-5)
        assert dl == pytest.approx(dr, abs=1e-4)
    # monotone decreasing, repulsive
    rs = np.linspace(0.05, 1.999, 400)
    us = np.array([oracle.zbl_pair(P, r)[0] for r in rs])
    assert np.all(np.diff(us) < 0) and np.all(us > 0)


def test_derivative_by_central_difference():
    P = _params()
    for r in (0.3, 0.8, 1.2, 1.5, 1.9):
        h = 1e-6
        fd = (oracle.zbl_pair(P, r + h)[0] - oracle.zbl_pair(P, r - h)[0]) / (2 * h)
        assert oracle.zbl_pair(P, r)[1] == pytest.approx(fd, rel=1e-7)


def test_dimer_energy_split_half_per_atom():
    # Eq. 1: each atom of an isolated dimer gets U_NEP + 1/2 U_ZBL; with a zero network the sum is U_ZBL.
    m = wl.synthetic_model()
    m["w1"] = np.zeros_like(m["w1"]); m["b1"] = 0.0
    P = oracle.Params(m)
    r = 1.37
    pos = np.array([[10.0, 10.0 + r], [10.0, 10.0], [10.0, 10.0]])
    res = oracle.compute(P, pos, None, np.diag([40.0, 40, 40]).ravel(), [0, 0, 0])
    u, du = oracle.zbl_pair(P, r)
    assert res.energy == pytest.approx([0.5 * u, 0.5 * u], rel=1e-14)
    # repulsive: atom 0 pushed to -x with magnitude |dU/dr|
    assert res.force[0] == pytest.approx([du, -du], rel=1e-13)
    assert np.all(res.force[1:] == 0)
    # virial: sum_i W_i^xx = -r dU/dr > 0 under compression
    assert res.virial[0].sum() == pytest.approx(-r * du, rel=1e-13)
