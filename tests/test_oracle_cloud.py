"""Pins for oracle/cloud.py (SURVEY.md 8(c) pins P5, P7 and the table invariants) -- CPU only.

Nothing here calls the oracle to check the oracle: the expected values are the paper's printed
numbers (tests/golden/paper_printed_values.txt), closed forms of the log-normal law, Gauss-Legendre
quadrature of the exact Mie function (numpy's nodes), and the definition of a quantile.
"""
import math
import os

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

import pdv_workloads as W
from oracle import cloud, mie

M_SN = complex(W.M_RE, W.M_IM)
LAM = W.WAVELENGTH


def _golden():
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_printed_values.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        name, val, tol = line.split()[:3]
        out[name] = (float(val), float(tol))
    return out


def _paper_cloud(m0_mg_cm2, d_m_um, sigma, n_classes=16):
    return cloud.build_cloud(W._cloud(m0_mg_cm2, 10.0, 2000.0, lognormal=(d_m_um, sigma, n_classes)),
                             phase_override=np.tile(np.linspace(-1, 1, 5), (n_classes, 1)))   # tables not needed


def test_paper_printed_optical_thickness_P7():
    """PAPER.md:373 prints tau0 = 23.4 and 8.6 with tau0 = g_back * 3 K_ext m0 / (2 rho0 d32) (Eq. 25-27),
    g_back = 0.67.  Pins Mie K_ext + log-normal classes + Eq. 10 in one number."""
    g = _golden()
    a = _paper_cloud(20.0, 1.5, 0.5, 600)          # finely resolved size law: the paper's own number
    b = _paper_cloud(10.0, 2.0, 0.5, 600)
    assert 0.67 * a.tau_ext == pytest.approx(g["tau0_case_a"][0], abs=g["tau0_case_a"][1])
    assert 0.67 * b.tau_ext == pytest.approx(g["tau0_case_b"][0], abs=g["tau0_case_b"][1])
    # the 16-class list of the boundary stays within 1.5 % of it
    assert 0.67 * _paper_cloud(20.0, 1.5, 0.5).tau_ext == pytest.approx(g["tau0_case_a"][0], rel=0.015)
    assert 0.67 * _paper_cloud(10.0, 2.0, 0.5).tau_ext == pytest.approx(g["tau0_case_b"][0], rel=0.015)


def test_paper_transport_thickness_weak_pin():
    """tau_tr = 10 <-> m0 = 10.7 mg/cm^2 (d_m = 1.5 um, sigma = 0.5); tau_tr = tau_ext (1 - omega0 g)."""
    g = _golden()
    c = _paper_cloud(10.7, 1.5, 0.5)
    om = float(np.sum(c.p_class * c.omega0))
    gbar = float(np.sum(c.p_class * c.omega0 * c.g) / np.sum(c.p_class * c.omega0))
    assert c.tau_ext * (1.0 - om * gbar) == pytest.approx(g["tau_tr_m0_10p7"][0], abs=g["tau_tr_m0_10p7"][1])


@pytest.mark.parametrize("sigma", [0.5, 0.7])
def test_lognormal_classes_moments(sigma):
    """Closed form of Eq. 21 (standard log-normal): <d^k> = d_m^k exp(k^2 sigma^2/2), hence the Sauter
    diameter d32 = d_m exp(2.5 sigma^2), which the paper prints.  16 classes on
    [-3, 3+3 sigma] reproduce it to a few per cent."""
    g = _golden()
    d, w = cloud.lognormal_classes(3e-6, sigma, 16)
    assert w.sum() == pytest.approx(1.0, abs=1e-14) and np.all(w > 0) and np.all(np.diff(d) > 0)
    d32 = np.sum(w * d**3) / np.sum(w * d**2)
    assert d32 / 3e-6 == pytest.approx(math.exp(g["sauter_factor_exp"][0] * sigma**2), rel=0.06)
    assert np.sum(w * d) / 3e-6 == pytest.approx(math.exp(0.5 * sigma**2), rel=0.03)
    # many classes converge to the closed form
    d, w = cloud.lognormal_classes(3e-6, sigma, 4000)
    assert np.sum(w * d**3) / np.sum(w * d**2) / 3e-6 == pytest.approx(math.exp(2.5 * sigma**2), rel=2e-3)


def test_monodisperse_limit():
    d, w = cloud.lognormal_classes(2e-6, 0.0, 16)
    assert d.tolist() == [2e-6] and w.tolist() == [1.0]


@pytest.mark.parametrize("d_um", [1.0, 5.0])
def test_phase_table_is_the_quantile_function_P5(d_um):
    """M[k] must satisfy F(M[k]) = k/K with F the CDF of |S1|^2+|S2|^2 in mu: checked by Gauss-Legendre
    quadrature of the exact Mie intensity (numpy nodes) between consecutive quantiles; plus monotone,
    end points, and table mean = Mie asymmetry g (series)."""
    x = math.pi * d_um * 1e-6 / LAM
    K = 1024
    M = cloud.phase_quantile_table(x, M_SN, K)
    assert M[0] == -1.0 and M[K] == 1.0 and np.all(np.diff(M) > 0)
    a, b = mie.coefficients(x, M_SN)
    ke, ks, ka, g = mie.efficiencies(x, M_SN)
    nodes, wts = npleg.leggauss(48)
    total = x * x * ks                                           # sum rule (pinned in test_oracle_mie)
    for k in (0, 1, 17, 400, 511, 900, K - 2, K - 1):
        lo, hi = M[k], M[k + 1]
        mu = 0.5 * (hi + lo) + 0.5 * (hi - lo) * nodes
        mass = 0.5 * (hi - lo) * np.sum(wts * mie.intensity(a, b, mu)) / total
        assert mass == pytest.approx(1.0 / K, rel=2e-5)
    assert np.sum(M[:-1] + M[1:]) / (2 * K) == pytest.approx(g, abs=2e-6)


def test_phase_table_backscatter_cone_probability():
    """Probability of the 0.1 sr backscatter cone (cos theta <= -mu_a) under D_1024 vs exact Mie."""
    x = math.pi * 5e-6 / LAM
    K = 1024
    M = cloud.phase_quantile_table(x, M_SN, K)
    mu_a = 1.0 - W.APERTURE_SR / (2 * math.pi)
    k = np.searchsorted(M, -mu_a) - 1
    p_table = (k + (-mu_a - M[k]) / (M[k + 1] - M[k])) / K
    a, b = mie.coefficients(x, M_SN)
    nodes, wts = npleg.leggauss(64)
    mu = 0.5 * (-mu_a - 1.0) + 0.5 * (1.0 - mu_a) * nodes
    p_exact = 0.5 * (1.0 - mu_a) * np.sum(wts * mie.intensity(a, b, mu)) / (x * x * mie.efficiencies(x, M_SN)[1])
    assert p_table == pytest.approx(p_exact, rel=5e-4)


def test_isotropic_table():
    M = cloud.isotropic_quantile_table(8)
    assert np.allclose(M, [-1, -0.75, -0.5, -0.25, 0, 0.25, 0.5, 0.75, 1])


def test_depth_table_closed_form(cfg2_oracle_cloud):
    """T(v) = tau_ext (1 - G(v)); G from Eq. 20 truncated to [v_fs, 3 v_fs] and renormalised: checked by
    quadrature of the printed density f(v) = (beta/v_fs) exp(-beta (v/v_fs - 1))."""
    c = cfg2_oracle_cloud
    n = c.T_edge.size - 1
    v_edges = c.v_max - (c.v_max - c.v_fs) * np.arange(n + 1) / n
    assert c.T_edge[0] == 0.0 and c.T_edge[-1] == c.tau_ext and np.all(np.diff(c.T_edge) > 0)
    f = lambda v: (c.beta / c.v_fs) * np.exp(-c.beta * (v / c.v_fs - 1.0))
    nodes, wts = npleg.leggauss(64)
    quad = lambda lo, hi: 0.5 * (hi - lo) * np.sum(wts * f(0.5 * (hi + lo) + 0.5 * (hi - lo) * nodes))
    total = quad(c.v_fs, c.v_max)
    for j in (1, 100, 512, 1000, n - 1):
        mass_above = quad(v_edges[j], c.v_max) / total            # mass between v_j and the top
        assert c.T_edge[j] == pytest.approx(c.tau_ext * mass_above, rel=1e-10)
    # mass-extinction coefficient, Eq. 10 for one diameter: kappa = 3 K_ext / (2 rho0 d)
    ke = mie.efficiencies(math.pi * 5e-6 / LAM, M_SN)[0]
    assert c.kappa == pytest.approx(3.0 * ke / (2.0 * W.DENSITY * 5e-6), rel=1e-12)
    assert c.tau_ext == pytest.approx(c.kappa * 2.0 * W.MG_CM2, rel=1e-12)


def test_class_probabilities_sum_and_weighting():
    c = _paper_cloud(20.0, 1.5, 0.5)
    assert c.p_class.sum() == pytest.approx(1.0, abs=1e-14)
    ref = c.number_weights * c.diameters**2 * c.k_ext
    assert np.allclose(c.p_class, ref / ref.sum(), rtol=1e-14)
    assert np.all((c.omega0 > 0.8) & (c.omega0 < 1.0))
