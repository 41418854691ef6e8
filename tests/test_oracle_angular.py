"""Pins of the oracle's angular descriptor and network (8(c) D).

The oracle uses Legendre double sums and Tr(S^3); here they are checked against the
spherical-harmonic forms built from library routines (scipy sph_harm_y, sympy wigner_3j),
closed forms for one neighbour, and symmetry zeros on cubic sites.
"""
import numpy as np
import pytest
from scipy.special import sph_harm_y

import oracle
from paper_2305_08140_b200 import workloads as wl

NR, NA, LMAX = 5, 5, 4


def _random_neighbourhood(seed, nn=11, rmin=1.2, rmax=5.8):
    g = wl.rng(seed, 9)
    v = g.standard_normal((nn, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    return v * g.uniform(rmin, rmax, size=(nn, 1))


def _angles(d):
    r = np.linalg.norm(d, axis=1)
    return r, np.arccos(d[:, 2] / r), np.arctan2(d[:, 1], d[:, 0])


def _A_nlm(P, d):
    """A_{n,l,m} = sum_j g^A_n(r_j) Y_lm(r_j), complex orthonormal Y_lm from scipy."""
    r, th, ph = _angles(d)
    A = {}
    for j in range(len(r)):
        if r[j] >= 4.0:
            continue
        g, _ = oracle.radial_functions(P, 1, r[j])
        for l in range(1, LMAX + 1):
            for m in range(-l, l + 1):
                A[(l, m)] = A.get((l, m), 0) + g * sph_harm_y(l, m, th[j], ph[j])
    return A


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_three_body_equals_sum_m_A_lm_squared(seed):
    # addition theorem: (2l+1)/(4pi) sum_jk g g P_l(cos) = sum_m |A_lm|^2
    P = oracle.Params(wl.synthetic_model())
    d = _random_neighbourhood(seed)
    q = oracle.descriptor_site(P, d)
    A = _A_nlm(P, d)
    for l in range(1, LMAX + 1):
        ref = sum(np.abs(A[(l, m)]) ** 2 for m in range(-l, l + 1))
        assert q[NR + (l - 1) * NA: NR + l * NA] == pytest.approx(ref, rel=1e-12, abs=1e-15)


@pytest.mark.parametrize("seed", [1, 2])
def test_four_body_equals_wigner_3j_contraction(seed):
    # q^{222}_n = sum_{m1 m2 m3} (2 2 2; m1 m2 m3) A_2m1 A_2m2 A_2m3  (SURVEY 8(c) C third bullet)
    from sympy.physics.wigner import wigner_3j
    P = oracle.Params(wl.synthetic_model())
    d = _random_neighbourhood(seed)
    q = oracle.descriptor_site(P, d)
    A = _A_nlm(P, d)
    ref = 0
    for m1 in range(-2, 3):
        for m2 in range(-2, 3):
            m3 = -m1 - m2
            if abs(m3) > 2:
                continue
            ref = ref + float(wigner_3j(2, 2, 2, m1, m2, m3)) * A[(2, m1)] * A[(2, m2)] * A[(2, m3)]
    assert np.abs(ref.imag).max() < 1e-14
    assert q[NR + LMAX * NA:] == pytest.approx(ref.real, rel=1e-11, abs=1e-16)


def test_four_body_constant_squared():
    # C^2 = 2025 / (896 pi^3)
    P = oracle.Params(wl.synthetic_model())
    d = np.array([[0.0, 0.0, 2.5]])
    g, _ = oracle.radial_functions(P, 1, 2.5)
    q = oracle.descriptor_site(P, d)
    C = q[NR + LMAX * NA:] / ((2.0 / 9.0) * g ** 3)     # single neighbour: Tr S^3 = (2/9) g^3
    assert C ** 2 == pytest.approx(np.full(NA, 2025 / (896 * np.pi ** 3)), rel=1e-13)
    assert np.all(C < 0)


def test_single_neighbour_closed_forms():
    # one neighbour at distance r, any direction: q_n = g^R_n, q_nl = (2l+1)/(4pi) g_n^2
    P = oracle.Params(wl.synthetic_model())
    for d in ([[1.1, -2.0, 1.7]], [[0.0, 3.0, 0.0]]):
        d = np.array(d)
        r = np.linalg.norm(d)
        q = oracle.descriptor_site(P, d)
        gR, _ = oracle.radial_functions(P, 0, r)
        gA, _ = oracle.radial_functions(P, 1, r)
        assert q[:NR] == pytest.approx(gR, rel=1e-14)
        for l in range(1, LMAX + 1):
            assert q[NR + (l - 1) * NA: NR + l * NA] == pytest.approx((2 * l + 1) / (4 * np.pi) * gA ** 2, rel=1e-13)
    # a neighbour between the two cutoffs contributes to the radial block only
    q = oracle.descriptor_site(P, np.array([[0.0, 0.0, 5.0]]))
    assert np.all(q[NR:] == 0) and np.any(q[:NR] != 0)


def test_cubic_site_symmetry_zeros():
    # perfect bcc site: A_lm = 0 for l = 1,2,3 and S = 0 (SURVEY 8(c) pins); l = 4 survives
    a = wl.A0_CONFIG
    pts = [np.array([i, j, k]) * a / 2 for i in range(-4, 5) for j in range(-4, 5) for k in range(-4, 5)
           if (i % 2 == j % 2 == k % 2) and (i, j, k) != (0, 0, 0)]
    d = np.array([p for p in pts if np.linalg.norm(p) < 6.0])
    assert len(d) == 58 and (np.linalg.norm(d, axis=1) < 4.0).sum() == 14
    P = oracle.Params(wl.synthetic_model())
    q = oracle.descriptor_site(P, d)
    assert np.abs(q[NR: NR + 3 * NA]).max() < 1e-13
    assert np.abs(q[NR + 4 * NA:]).max() < 1e-15
    assert np.abs(q[NR + 3 * NA: NR + 4 * NA]).min() > 1e-6


def test_descriptor_is_rotation_and_order_invariant():
    P = oracle.Params(wl.synthetic_model())
    d = _random_neighbourhood(5, nn=14)
    q = oracle.descriptor_site(P, d)
    g = wl.rng(5, 10)
    R, _ = np.linalg.qr(g.standard_normal((3, 3)))
    q_rot = oracle.descriptor_site(P, d @ R.T)
    q_perm = oracle.descriptor_site(P, d[g.permutation(len(d))])
    assert q_rot == pytest.approx(q, rel=1e-11, abs=1e-14)
    assert q_perm == pytest.approx(q, rel=1e-12, abs=1e-15)


def test_descriptor_derivative_by_central_difference():
    P = oracle.Params(wl.synthetic_model())
    d = _random_neighbourhood(7, nn=9, rmax=5.0)
    q, dq = oracle.descriptor_site(P, d, want_dq=True)
    h = 1e-6
    for j in range(len(d)):
        for a in range(3):
            dp = d.copy(); dp[j, a] += h
            dm = d.copy(); dm[j, a] -= h
            fd = (oracle.descriptor_site(P, dp) - oracle.descriptor_site(P, dm)) / (2 * h)
            assert dq[:, j, a] == pytest.approx(fd, rel=2e-6, abs=1e-9)


def test_network_hand_computed_and_gradient():
    # D = 2 (n_max_R = 1, no angular part), one neuron: U = w1 tanh(w00 s0 q0 + w01 s1 q1 - b0) - b1
    m = wl.synthetic_model(n_max_radial=1, n_max_angular=-1, l_max=0, has_4body=0, n_neurons=1)
    m.update(w0=[[0.3, -0.7]], b0=[0.1], w1=[1.5], b1=0.25, q_scaler=[2.0, 0.5])
    P = oracle.Params(m)
    assert P.D == 2
    q = np.array([0.4, -1.2])
    U, Fp = oracle.site_energy(P, q)
    z = 0.3 * 2.0 * 0.4 + (-0.7) * 0.5 * (-1.2) - 0.1
    assert U == pytest.approx(1.5 * np.tanh(z) - 0.25, rel=1e-15)
    sech2 = 1 - np.tanh(z) ** 2
    assert Fp == pytest.approx([1.5 * sech2 * 0.3 * 2.0, 1.5 * sech2 * (-0.7) * 0.5], rel=1e-14)
    # full-size network: dU/dq against central differences
    P = oracle.Params(wl.synthetic_model())
    q = wl.rng(3, 11).standard_normal(P.D) * 0.5
    U, Fp = oracle.site_energy(P, q)
    for v in range(P.D):
        e = np.zeros(P.D); e[v] = 1e-6
        fd = (oracle.site_energy(P, q + e)[0] - oracle.site_energy(P, q - e)[0]) / 2e-6
        assert Fp[v] == pytest.approx(fd, rel=1e-7, abs=1e-9)


# ------------------------------------------------------------------ 5-body term (C-27)

def _five_body_model():
    return wl.synthetic_model(has_5body=1)


@pytest.mark.parametrize("seed", [1, 2])
def test_five_body_equals_wigner_3j_contraction(seed):
    # q^{1111}_n = sum_{m1..m4} (1 1 0; m1 m2 0)(1 1 0; m3 m4 0) A_1m1 A_1m2 A_1m3 A_1m4 with orthonormal complex Y_1m:
    # the library 3j symbols and spherical harmonics against the oracle's quadruple sum over neighbours
    from sympy.physics.wigner import wigner_3j
    P = oracle.Params(_five_body_model())
    assert P.D == 35
    d = _random_neighbourhood(seed)
    q = oracle.descriptor_site(P, d)
    A = _A_nlm(P, d)
    pair = 0
    for m1 in (-1, 0, 1):
        pair = pair + float(wigner_3j(1, 1, 0, m1, -m1, 0)) * A[(1, m1)] * A[(1, -m1)]
    ref = pair * pair
    assert np.abs(ref.imag).max() < 1e-14
    assert q[NR + (LMAX + 1) * NA:] == pytest.approx(ref.real, rel=1e-11, abs=1e-18)
    # and, by the addition theorem, one third of the squared l = 1 three-body component
    assert q[NR + (LMAX + 1) * NA:] == pytest.approx(q[NR:NR + NA] ** 2 / 3.0, rel=1e-12, abs=1e-18)


def test_five_body_single_neighbour_cubic_site_and_derivative():
    P = oracle.Params(_five_body_model())
    r = 2.7
    g, _ = oracle.radial_functions(P, 1, r)
    q = oracle.descriptor_site(P, np.array([[0.0, r, 0.0]]))
    assert q[30:] == pytest.approx((3.0 / (4 * np.pi) * g ** 2) ** 2 / 3.0, rel=1e-13)      # one neighbour: v.v = g^2
    a = wl.A0_CONFIG                                                                          # cubic site: sum_j v_j = 0
    pts = np.array([[i, j, k] for i in (-1, 1) for j in (-1, 1) for k in (-1, 1)]) * a / 2
    assert np.abs(oracle.descriptor_site(P, pts)[30:]).max() < 1e-18      # rounding of the cancelling quadruple sum
    d = _random_neighbourhood(7, nn=9, rmax=5.0)
    q, dq = oracle.descriptor_site(P, d, want_dq=True)
    h = 1e-6
    for j in range(len(d)):
        for a_ in range(3):
            dp = d.copy(); dp[j, a_] += h
            dm = d.copy(); dm[j, a_] -= h
            fd = (oracle.descriptor_site(P, dp) - oracle.descriptor_site(P, dm)) / (2 * h)
            assert dq[30:, j, a_] == pytest.approx(fd[30:], rel=2e-6, abs=1e-12)
