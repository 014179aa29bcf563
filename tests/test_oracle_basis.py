"""Pins for the oracle's Chebyshev basis and cutoff (paper App.A; Eq.6)."""
import numpy as np
import pytest

from oracle import gnep_oracle as orc


def _Tk(rc, K, d):
    f, _ = orc.basis(rc, K, d)
    fc = 0.5 * (1 + np.cos(np.pi * d / rc))
    return 2 * f / fc - 1


def test_chebyshev_is_cos_k_phi():
    rc, K = 6.0, 12
    for d in np.linspace(0.3, 5.7, 23):
        xi = 2 * (d / rc - 1) ** 2 - 1
        phi = np.arccos(xi)
        np.testing.assert_allclose(_Tk(rc, K, d), np.cos(np.arange(K) * phi), atol=1e-12)


def test_chebyshev_end_values_and_derivative_at_one():
    rc, K = 5.0, 10
    # d -> 0: xi = 1: T_k = 1 so f_k(0) = 1
    f, fp = orc.basis(rc, K, 0.0)
    np.testing.assert_allclose(f, np.ones(K), atol=1e-14)
    # xi = -1 at d = rc(1 - 1/sqrt 2)... use x^2 = 0 -> d = rc is the cutoff; instead check T_k(-1) at xi=-1: d = rc
    # T_k'(1) = k^2: fp(0) = 1/2 T_k'(1) dxi/dd f_c + (T_k+1)/2 f_c' ; at d=0 f_c'=0, f_c=1, dxi/dd = -4/rc
    np.testing.assert_allclose(fp, 0.5 * np.arange(K) ** 2 * (-4.0 / rc), atol=1e-12)
    # at x = 0 (d = rc) xi = -1: T_k = (-1)^k, but f_c = 0 -> f = 0
    d = rc * (1 - 1e-9)
    f, _ = orc.basis(rc, K, d)
    assert np.all(np.abs(f) < 1e-15)


def test_smooth_cutoff():
    """f_k and f_k' vanish at r_c and beyond."""
    for rc, K in ((4.0, 6), (8.0, 12)):
        for d in (rc, rc * 1.1):
            f, fp = orc.basis(rc, K, d)
            assert np.all(np.abs(f) < 1e-15) and np.all(np.abs(fp) < 1e-15)
        f, fp = orc.basis(rc, K, rc * (1 - 1e-7))
        assert np.all(np.abs(f) < 1e-12) and np.all(np.abs(fp) < 1e-5)


def test_basis_derivative_fd():
    rc, K, h = 7.0, 12, 1e-6
    for d in (0.5, 2.2, 3.5, 5.1, 6.9):
        _, fp = orc.basis(rc, K, d)
        fd = (orc.basis(rc, K, d + h)[0] - orc.basis(rc, K, d - h)[0]) / (2 * h)
        np.testing.assert_allclose(fp, fd, rtol=0, atol=2e-8)


def test_basis_bounded():
    """0 <= f_k <= 1 because |T_k| <= 1 and 0 <= f_c <= 1."""
    for d in np.linspace(0, 6, 50):
        f, _ = orc.basis(6.0, 16, d)
        assert np.all(f >= -1e-15) and np.all(f <= 1 + 1e-15)
