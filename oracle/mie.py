"""ORACLE (test infrastructure, fp64) -- Mie theory for a homogeneous sphere, Eq. 12-14.

This file is part of `oracle/`: a plain, slow, double-precision CPU restatement of the paper's
method.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import it.  It shares no code with the CUDA library (paper_2012_00963_b200/csrc) and never
imports it.

What is computed, with the passage that defines it:

* size parameter alpha = pi d / lambda
* K_ext = (2/alpha^2) sum (2n+1) Re(a_n + b_n)                           Eq. 12
  K_sca = (2/alpha^2) sum (2n+1) (|a_n|^2 + |b_n|^2),  K_abs = K_ext - K_sca
* S1 = sum (2n+1)/(n(n+1)) (a_n pi_n + b_n tau_n), S2 with pi/tau swapped Eq. 14
  with pi_n = dP_n(cos th)/dcos th and tau_n = dP_n^(1)(cos th)/dth, as the paper writes them.
* unpolarised phase function p(th) proportional to |S1|^2 + |S2|^2       Eq. 13
  (normalised numerically: the printed prefactor lambda^2/(2 pi K_sca) is dimensionally loose,
  DESIGN.md reading R9).

The paper does not print a_n, b_n ("Mie coefficients", ref. 33).  They are the textbook ones for a
non-magnetic sphere of relative index m (time factor exp(-i w t), so Im m > 0 absorbs):

    a_n = [ (D_n(mx)/m + n/x) psi_n(x) - psi_{n-1}(x) ] / [ (D_n(mx)/m + n/x) xi_n(x) - xi_{n-1}(x) ]
    b_n = [ (m D_n(mx) + n/x) psi_n(x) - psi_{n-1}(x) ] / [ (m D_n(mx) + n/x) xi_n(x) - xi_{n-1}(x) ]

psi_n(x) = x j_n(x), xi_n(x) = x (j_n(x) + i y_n(x)), D_n(z) = psi_n'(z)/psi_n(z).
psi_n, xi_n come from scipy's spherical Bessel routines (library primitive, real argument);
D_n(mx) from the downward recurrence D_{n-1} = n/z - 1/(D_n + n/z), which never overflows for the
strongly absorbing index used here.

Pins (tests/test_oracle_mie.py): the a_n, b_n above against the Wronskian-ratio textbook formula
evaluated with scipy/mpmath complex spherical Bessel functions; Rayleigh limit; K_ext -> 2 at large
x; sum rule  int(|S1|^2+|S2|^2) dmu = x^2 K_sca; g series against quadrature; pi_n/tau_n against
numpy's Legendre polynomials.
"""
from __future__ import annotations

import math

import numpy as np
from scipy import special


def n_terms(x: float) -> int:
    """Series truncation n_max = ceil(x + 4 x^(1/3) + 2) (standard)."""
    return int(math.ceil(x + 4.0 * x ** (1.0 / 3.0) + 2.0))


def log_derivative(z: complex, n_max: int) -> np.ndarray:
    """D_n(z) = psi_n'(z)/psi_n(z) for n = 0..n_max by downward recurrence from D = 0 far above n_max."""
    n_start = int(max(n_max, abs(z))) + 16
    D = np.zeros(n_start + 1, dtype=np.complex128)
    for n in range(n_start, 0, -1):
        D[n - 1] = n / z - 1.0 / (D[n] + n / z)
    return D[: n_max + 1]


def coefficients(x: float, m: complex, n_max: int | None = None):
    """Mie coefficients a_n, b_n for n = 1..n_max (arrays indexed n-1)."""
    if n_max is None:
        n_max = n_terms(x)
    n = np.arange(0, n_max + 1)
    jn = special.spherical_jn(n, x)
    yn = special.spherical_yn(n, x)
    psi = x * jn
    xi = x * (jn + 1j * yn)
    D = log_derivative(m * x, n_max)
    nn = n[1:]
    ta = D[1:] / m + nn / x
    tb = D[1:] * m + nn / x
    a = (ta * psi[1:] - psi[:-1]) / (ta * xi[1:] - xi[:-1])
    b = (tb * psi[1:] - psi[:-1]) / (tb * xi[1:] - xi[:-1])
    return a, b


def efficiencies(x: float, m: complex):
    """(K_ext, K_sca, K_abs, g) of Eq. 12; g is the asymmetry parameter <cos theta> (series form)."""
    a, b = coefficients(x, m)
    n = np.arange(1, len(a) + 1)
    k_ext = (2.0 / x**2) * np.sum((2 * n + 1) * (a + b).real)
    k_sca = (2.0 / x**2) * np.sum((2 * n + 1) * (np.abs(a) ** 2 + np.abs(b) ** 2))
    s = np.sum((2 * n + 1) / (n * (n + 1.0)) * (a * np.conj(b)).real)
    s += np.sum((n[:-1] * (n[:-1] + 2.0) / (n[:-1] + 1.0)) * (a[:-1] * np.conj(a[1:]) + b[:-1] * np.conj(b[1:])).real)
    g = (4.0 / (x**2 * k_sca)) * s
    return float(k_ext), float(k_sca), float(k_ext - k_sca), float(g)


def pi_tau(mu: np.ndarray, n_max: int):
    """Angular functions pi_n = dP_n/dmu and tau_n = dP_n^(1)/dtheta, n = 1..n_max, shape (n_max, len(mu)).

    Upward recurrences (textbook): pi_0 = 0, pi_1 = 1,
    pi_n = ((2n-1)/(n-1)) mu pi_{n-1} - (n/(n-1)) pi_{n-2},   tau_n = n mu pi_n - (n+1) pi_{n-1}.
    """
    mu = np.asarray(mu, dtype=np.float64)
    pi = np.zeros((n_max + 1, mu.size))
    tau = np.zeros((n_max + 1, mu.size))
    pi[1] = 1.0
    tau[1] = mu
    for n in range(2, n_max + 1):
        pi[n] = ((2 * n - 1) / (n - 1.0)) * mu * pi[n - 1] - (n / (n - 1.0)) * pi[n - 2]
        tau[n] = n * mu * pi[n] - (n + 1) * pi[n - 1]
    return pi[1:], tau[1:]


def amplitudes(a: np.ndarray, b: np.ndarray, mu: np.ndarray):
    """S1(theta), S2(theta) of Eq. 14 at mu = cos(theta)."""
    n_max = len(a)
    pi, tau = pi_tau(mu, n_max)
    n = np.arange(1, n_max + 1)
    f = (2 * n + 1) / (n * (n + 1.0))
    s1 = (f * a) @ pi + (f * b) @ tau
    s2 = (f * a) @ tau + (f * b) @ pi
    return s1, s2


def intensity(a: np.ndarray, b: np.ndarray, mu: np.ndarray) -> np.ndarray:
    """|S1|^2 + |S2|^2: the unnormalised unpolarised phase function of Eq. 13."""
    s1, s2 = amplitudes(a, b, mu)
    return np.abs(s1) ** 2 + np.abs(s2) ** 2
