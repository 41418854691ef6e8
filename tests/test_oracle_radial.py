"""Pins of the oracle's radial functions (Chebyshev basis, cutoffs P:106)."""
import numpy as np
import pytest

import oracle
from paper_2305_08140_b200 import workloads as wl


def test_chebyshev_identity_T_k_cos_theta():
    # f_k(r) = 1/2 [T_k(x)+1] f_c(r): recover T_k and check T_k(cos t) = cos(k t)
    rc, basis = 6.0, 12
    for r in np.linspace(0.1, 5.9, 25):
        f, _ = oracle.radial_basis(r, rc, basis)
        fc = 0.5 * (1 + np.cos(np.pi * r / rc))
        x = 2 * (r / rc - 1) ** 2 - 1
        T = 2 * f / fc - 1
        assert T == pytest.approx(np.cos(np.arange(basis + 1) * np.arccos(x)), abs=1e-12)


def test_special_values():
    rc, basis = 4.0, 8
    f, df = oracle.radial_basis(rc, rc, basis)
    assert np.all(f == 0) and np.all(df == 0)            # zero at and beyond the cutoff
    f, df = oracle.radial_basis(rc * (1 - 1e-9), rc, basis)
    assert np.all(np.abs(f) < 1e-15) and np.all(np.abs(df) < 1e-7)   # C^1 at the cutoff
    f, _ = oracle.radial_basis(1e-13, rc, basis)         # r -> 0: x = 1, T_k = 1, f_c = 1
    assert f == pytest.approx(np.ones(basis + 1), abs=1e-10)
    f, _ = oracle.radial_basis(rc / 2, rc, basis)        # f_0 = f_c = 1/2 at rc/2
    assert f[0] == pytest.approx(0.5, abs=1e-15)
    # at r = rc(1 - 1/sqrt 2): x = 0, so T_k = cos(k pi/2)
    r = rc * (1 - 1 / np.sqrt(2))
    f, _ = oracle.radial_basis(r, rc, basis)
    fc = 0.5 * (1 + np.cos(np.pi * r / rc))
    assert 2 * f / fc - 1 == pytest.approx(np.cos(np.arange(basis + 1) * np.pi / 2), abs=1e-12)


def test_derivative_by_central_difference():
    rc, basis = 6.0, 8
    for r in (0.4, 1.7, 3.3, 5.2, 5.95):
        h = 1e-6
        fp, _ = oracle.radial_basis(r + h, rc, basis)
        fm, _ = oracle.radial_basis(r - h, rc, basis)
        _, df = oracle.radial_basis(r, rc, basis)
        assert df == pytest.approx((fp - fm) / (2 * h), rel=1e-7, abs=1e-9)


@pytest.mark.parametrize("which", [0, 1])
def test_g_n_reduces_to_f_n_for_identity_coefficients(which):
    m = wl.synthetic_model()
    key = "c_angular" if which else "c_radial"
    c = np.zeros_like(m[key])
    for n in range(c.shape[2]):
        c[0, 0, n, n] = 1.0
    m[key] = c
    P = oracle.Params(m)
    rc = m["rc_angular"] if which else m["rc_radial"]
    for r in (0.9, 2.5, 3.9):
        g, dg = oracle.radial_functions(P, which, r)
        f, df = oracle.radial_basis(r, rc, 8)
        assert g == pytest.approx(f[:5], abs=1e-15)
        assert dg == pytest.approx(df[:5], abs=1e-15)


def test_g_n_is_the_coefficient_contraction_and_uses_own_cutoff():
    m = wl.synthetic_model()
    P = oracle.Params(m)
    r = 3.1
    for which, rc, key in ((0, 6.0, "c_radial"), (1, 4.0, "c_angular")):
        g, _ = oracle.radial_functions(P, which, r)
        f, _ = oracle.radial_basis(r, rc, 8)
        assert g == pytest.approx(m[key][0, 0] @ f, abs=1e-14)
    assert np.all(oracle.radial_functions(P, 1, 4.5)[0] == 0)      # beyond the angular cutoff
    assert np.any(oracle.radial_functions(P, 0, 4.5)[0] != 0)      # but inside the radial one


def test_type_pair_coefficients_are_indexed_ti_tj():
    m = wl.synthetic_model(n_types=2)
    P = oracle.Params(m)
    f, _ = oracle.radial_basis(2.2, 6.0, 8)
    for ti in range(2):
        for tj in range(2):
            g, _ = oracle.radial_functions(P, 0, 2.2, ti, tj)
            assert g == pytest.approx(m["c_radial"][ti, tj] @ f, abs=1e-14)
