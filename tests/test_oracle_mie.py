"""Pins for oracle/mie.py (SURVEY.md 8(c) pins P4, P5) -- CPU only.

Each test checks the oracle against something other than itself: the textbook Wronskian-ratio
definition of a_n, b_n evaluated with library Bessel functions (scipy, mpmath), the Rayleigh and
geometric-optics limits, the optical-theorem style sum rule tying Eq. 14 to Eq. 12, and numpy's
Legendre polynomials for pi_n / tau_n.
"""
import math

import mpmath
import numpy as np
import pytest
from numpy.polynomial import legendre as npleg
from scipy import special

from oracle import mie

M_SN = complex(2.5, 9.5)
LAM = 1550e-9


def _textbook_ab_scipy(x, m, n_max):
    """a_n, b_n from the textbook definition (Bohren & Huffman Eq. 4.53) with complex Bessel functions."""
    n = np.arange(1, n_max + 1)
    z = m * x
    psi = lambda t, nn: t * special.spherical_jn(nn, t)
    dpsi = lambda t, nn: special.spherical_jn(nn, t) + t * special.spherical_jn(nn, t, derivative=True)
    xi = lambda t, nn: t * (special.spherical_jn(nn, t) + 1j * special.spherical_yn(nn, t))
    dxi = lambda t, nn: (special.spherical_jn(nn, t) + 1j * special.spherical_yn(nn, t)) + t * (
        special.spherical_jn(nn, t, derivative=True) + 1j * special.spherical_yn(nn, t, derivative=True))
    a = (m * psi(z, n) * dpsi(x, n) - psi(x, n) * dpsi(z, n)) / (m * psi(z, n) * dxi(x, n) - xi(x, n) * dpsi(z, n))
    b = (psi(z, n) * dpsi(x, n) - m * psi(x, n) * dpsi(z, n)) / (psi(z, n) * dxi(x, n) - m * xi(x, n) * dpsi(z, n))
    return a, b


@pytest.mark.parametrize("d_um", [1.0, 2.0, 5.0, 10.0])
def test_coefficients_match_textbook_definition_scipy(d_um):
    x = math.pi * d_um * 1e-6 / LAM
    a, b = mie.coefficients(x, M_SN)
    a2, b2 = _textbook_ab_scipy(x, M_SN, len(a))
    assert np.allclose(a, a2, rtol=1e-9, atol=1e-13)
    assert np.allclose(b, b2, rtol=1e-9, atol=1e-13)


def test_coefficients_match_mpmath_high_precision():
    """30-digit evaluation of the same definition for a dielectric-ish and the tin index."""
    mpmath.mp.dps = 30
    for x, m in ((3.7, complex(1.5, 0.01)), (10.134169850289657, M_SN)):
        a, b = mie.coefficients(x, m)
        mm, xx = mpmath.mpc(m), mpmath.mpf(x)
        sj = lambda n, t: mpmath.sqrt(mpmath.pi / (2 * t)) * mpmath.besselj(n + 0.5, t)
        sy = lambda n, t: mpmath.sqrt(mpmath.pi / (2 * t)) * mpmath.bessely(n + 0.5, t)
        for n in (1, 2, 5, len(a) - 2):
            psi = lambda t: t * sj(n, t)
            xi = lambda t: t * (sj(n, t) + 1j * sy(n, t))
            dpsi = lambda t: mpmath.diff(psi, t)
            dxi = lambda t: mpmath.diff(xi, t)
            z = mm * xx
            an = (mm * psi(z) * dpsi(xx) - psi(xx) * dpsi(z)) / (mm * psi(z) * dxi(xx) - xi(xx) * dpsi(z))
            bn = (psi(z) * dpsi(xx) - mm * psi(xx) * dpsi(z)) / (psi(z) * dxi(xx) - mm * xi(xx) * dpsi(z))
            assert abs(complex(an) - a[n - 1]) < 1e-10 * max(1.0, abs(a[n - 1])) + 1e-14
            assert abs(complex(bn) - b[n - 1]) < 1e-10 * max(1.0, abs(b[n - 1])) + 1e-14


def test_rayleigh_limit():
    """x -> 0:  K_sca = (8/3) x^4 |(m^2-1)/(m^2+2)|^2,  K_abs = 4 x Im((m^2-1)/(m^2+2))."""
    m = complex(1.6, 0.2)
    x = 1e-3
    ke, ks, ka, g = mie.efficiencies(x, m)
    L = (m * m - 1) / (m * m + 2)
    assert ks == pytest.approx((8.0 / 3.0) * x**4 * abs(L) ** 2, rel=1e-4)
    assert ka == pytest.approx(4.0 * x * L.imag, rel=1e-4)
    assert abs(g) < 1e-4


def test_large_sphere_extinction_paradox_and_absorption_sign():
    """K_ext -> 2 for x >> 1; Im(m) > 0 absorbs (K_abs > 0); p_s + p_a = 1."""
    excess = [mie.efficiencies(x, M_SN)[0] - 2.0 for x in (50.0, 100.0, 400.0, 1000.0)]
    assert all(e > 0 for e in excess) and excess == sorted(excess, reverse=True)   # edge term ~ x^(-2/3) decays
    assert excess[-1] < 0.05
    for d_um in (1, 2, 5, 10):
        ke, ks, ka, g = mie.efficiencies(math.pi * d_um * 1e-6 / LAM, M_SN)
        assert ka > 0 and ks > 0 and ks / ke + ka / ke == pytest.approx(1.0, abs=1e-15)


def test_non_absorbing_sphere_conserves():
    ke, ks, ka, g = mie.efficiencies(5.0, complex(1.33, 0.0))
    assert ka == pytest.approx(0.0, abs=1e-12)


def test_survey_reference_values_5um():
    """SURVEY.md 8(c) P4 quotes (est.) K_ext=2.2688, K_sca=2.1102, g=0.5371 for d = 5 um."""
    ke, ks, ka, g = mie.efficiencies(math.pi * 5e-6 / LAM, M_SN)
    assert ke == pytest.approx(2.2688, abs=5e-4)
    assert ks == pytest.approx(2.1102, abs=5e-4)
    assert g == pytest.approx(0.5371, abs=5e-4)


def test_pi_tau_against_numpy_legendre():
    """pi_n = dP_n/dmu, tau_n = dP_n^1/dtheta = mu pi_n - (1-mu^2) dpi_n/dmu."""
    mu = np.array([-0.97, -0.3, 0.0, 0.41, 0.999])
    n_max = 12
    pi, tau = mie.pi_tau(mu, n_max)
    for n in range(1, n_max + 1):
        c = np.zeros(n + 1)
        c[n] = 1.0
        d1 = npleg.legval(mu, npleg.legder(c, 1))
        d2 = npleg.legval(mu, npleg.legder(c, 2)) if n >= 2 else np.zeros_like(mu)
        assert np.allclose(pi[n - 1], d1, rtol=1e-12, atol=1e-12)
        assert np.allclose(tau[n - 1], mu * d1 - (1 - mu**2) * d2, rtol=1e-11, atol=1e-11)


@pytest.mark.parametrize("d_um", [1.0, 5.0, 10.0])
def test_sum_rule_and_asymmetry_by_quadrature(d_um):
    """int_{-1}^{1} (|S1|^2+|S2|^2) dmu = x^2 K_sca ties Eq. 14 to Eq. 12 (P5); g series = <mu>."""
    x = math.pi * d_um * 1e-6 / LAM
    a, b = mie.coefficients(x, M_SN)
    ke, ks, ka, g = mie.efficiencies(x, M_SN)
    nodes, wts = npleg.leggauss(400)
    I = mie.intensity(a, b, nodes)
    assert np.sum(wts * I) == pytest.approx(x * x * ks, rel=1e-10)
    assert np.sum(wts * I * nodes) / np.sum(wts * I) == pytest.approx(g, abs=1e-10)


def test_forward_and_backward_amplitudes():
    """S1(0) = S2(0) = (1/2) sum (2n+1)(a_n+b_n) (optical theorem: K_ext = 4 Re S(0)/x^2); S1(pi) = -S2(pi)."""
    x = math.pi * 5e-6 / LAM
    a, b = mie.coefficients(x, M_SN)
    s1, s2 = mie.amplitudes(a, b, np.array([1.0, -1.0]))
    n = np.arange(1, len(a) + 1)
    assert s1[0] == pytest.approx(0.5 * np.sum((2 * n + 1) * (a + b)), rel=1e-12)
    assert s2[0] == pytest.approx(s1[0], rel=1e-12)
    assert s1[1] == pytest.approx(-s2[1], rel=1e-10)
    ke = mie.efficiencies(x, M_SN)[0]
    assert ke == pytest.approx(4.0 * s1[0].real / x**2, rel=1e-12)
