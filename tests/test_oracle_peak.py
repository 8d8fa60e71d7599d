"""Pins for oracle/peak.py (readings R27-R30) -- CPU only.

Expected values are the paper's closed forms for the single-scattering spectrum Eq. 28 (peak position Eq. 31, peak
value Eq. 32, relative curvature Eq. 34), an exact parabola, and numpy's own convolution.
"""
import math

import numpy as np
import pytest

from oracle import peak

N = 10 ** 9


def _hist_from_cdf(F, n_bins, v_lo, v_hi, v_fs):
    """N * (F(x_{k+1}) - F(x_k)) for the bin edges x_k = (v_lo + k dv) / v_fs."""
    edges = (v_lo + np.arange(n_bins + 1) * (v_hi - v_lo) / n_bins) / v_fs
    return N * np.diff(F(edges))


@pytest.mark.parametrize("beta,tau0", [(10.0, 23.4), (6.0, 8.6), (14.0, 23.4)])
def test_peak_of_the_single_scattering_spectrum_Eq31_32_34(beta, tau0):
    """Eq. 28 in x = v/v_fs with f(x) = beta exp(-beta (x - 1)) (Eq. 20 as a density in x):
    I(x) = tau0 f exp(-tau0 f / beta) has the antiderivative exp(-tau0 f / beta), its peak at
    x = 1 + ln(tau0)/beta (Eq. 31), the peak value beta / e (Eq. 32: proportional to beta) and the relative curvature
    -beta^2 (Eq. 34).  tau0 = 23.4 and 8.6 are the paper's two cases."""
    v_fs, v_lo, v_hi, n_bins = 2000.0, 0.0, 6000.0, 4096
    F = lambda x: np.exp(-tau0 * beta * np.exp(-beta * (x - 1.0)) / beta)
    hist = _hist_from_cdf(F, n_bins, v_lo, v_hi, v_fs)
    r = peak.spectrum_peak(hist, N, v_lo, v_hi, v_fs, half=2, n_pass=1, fit_half=8, x_min=1.02)
    assert r["status"] == 0
    assert r["x_peak"] == pytest.approx(1.0 + math.log(tau0) / beta, abs=2e-4)
    assert r["i_peak"] == pytest.approx(beta / math.e, rel=2e-3)
    assert r["curvature"] == pytest.approx(-beta * beta, rel=2e-2)


def test_exact_parabola_is_recovered():
    """Point samples of A - C (x - x0)^2 at the bin centres: the least-squares parabola is that parabola."""
    v_fs, v_lo, v_hi, n_bins = 2000.0, 0.0, 6000.0, 512
    A, C, x0 = 3.0, 40.0, 1.3337
    dx = (v_hi - v_lo) / n_bins / v_fs
    x = (v_lo + (np.arange(n_bins) + 0.5) * (v_hi - v_lo) / n_bins) / v_fs
    hist = np.maximum(A - C * (x - x0) ** 2, 0.0) * N * dx
    r = peak.spectrum_peak(hist, N, v_lo, v_hi, v_fs, half=3, n_pass=2, fit_half=10, x_min=1.02)
    assert r["status"] == 0
    assert r["x_peak"] == pytest.approx(x0, abs=1e-10)
    assert r["i_peak"] == pytest.approx(A, rel=1e-10)
    assert r["curvature"] == pytest.approx(-2.0 * C / A, rel=1e-9)
    assert abs(x[r["k_peak"]] - x0) <= dx                      # the arg-max bin is the one next to the vertex


def test_moving_average_against_numpy_convolution_and_at_the_ends():
    rng = np.random.default_rng(5)
    s = rng.random(200)
    for half in (1, 4, 7):
        out = peak.moving_average(s, half)
        ref = np.convolve(s, np.ones(2 * half + 1) / (2 * half + 1), mode="valid")
        assert np.allclose(out[half:-half], ref, rtol=0, atol=1e-14)
        assert out[0] == pytest.approx(np.mean(s[:half + 1]))                 # truncated windows: mean of what exists
        assert out[-1] == pytest.approx(np.mean(s[-(half + 1):]))
        assert out[1] == pytest.approx(np.mean(s[:half + 2]))
    assert np.allclose(peak.moving_average(np.full(50, 2.5), 6), 2.5)         # a constant stays a constant
    ramp = np.arange(60.0)
    assert np.allclose(peak.moving_average(ramp, 5)[5:-5], ramp[5:-5])        # symmetric window: a ramp too


def test_search_range_skips_the_free_surface_peak_and_ties_take_the_first_bin():
    """Thin clouds show a second, larger peak at the free surface; x_min keeps it out (R28)."""
    v_fs, v_lo, v_hi, n_bins = 2000.0, 0.0, 6000.0, 600
    x = (np.arange(n_bins) + 0.5) * 0.005
    dx = 0.005
    s = 5.0 * np.exp(-0.5 * ((x - 0.99) / 0.01) ** 2) + 1.0 * np.exp(-0.5 * ((x - 1.5) / 0.1) ** 2)
    hist = s * N * dx
    r = peak.spectrum_peak(hist, N, v_lo, v_hi, v_fs, half=2, n_pass=1, fit_half=6, x_min=1.05)
    assert r["status"] == 0 and r["x_peak"] == pytest.approx(1.5, abs=2e-3)
    # Gaussian: I''/I = -1/sigma^2 at the top; a parabola over +-0.3 sigma sees the quartic term: -2.3 %
    assert r["curvature"] == pytest.approx(-1.0 / 0.1 ** 2, rel=0.03)
    r0 = peak.spectrum_peak(hist, N, v_lo, v_hi, v_fs, half=2, n_pass=1, fit_half=2, x_min=0.0)
    assert r0["x_peak"] == pytest.approx(0.99, abs=2e-3)
    flat = np.zeros(n_bins)
    flat[300:310] = 7.0                                                       # plateau: smoothed maximum is flat over bins 302..307
    rt = peak.spectrum_peak(flat, N, v_lo, v_hi, v_fs, half=2, n_pass=1, fit_half=1, x_min=0.0)
    assert rt["k_peak"] == 302                                                # the first of the tied bins


def test_status_codes():
    v_fs, v_lo, v_hi = 2000.0, 0.0, 6000.0
    z = peak.spectrum_peak(np.ones(64), N, v_lo, v_hi, v_fs, x_min=5.0)        # nothing in the search range
    assert z["status"] == 1 and z["k_peak"] == -1
    two = peak.spectrum_peak(np.array([1.0, 2.0]), N, v_lo, v_hi, v_fs, x_min=0.0, half=0, n_pass=0, fit_half=4)
    assert two["status"] == 1 and two["k_peak"] == 1
    cup = peak.spectrum_peak((np.arange(64.0) - 40) ** 2 + 1, N, v_lo, v_hi, v_fs, x_min=0.0, x_max=1.0, half=0,
                             n_pass=0, fit_half=3)                             # convex everywhere: c > 0
    assert cup["status"] == 2 and cup["curvature"] == 0.0
    empty = peak.spectrum_peak(np.zeros(32), 0, v_lo, v_hi, v_fs, x_min=0.0)   # n_photons = 0: zero spectrum
    assert empty["status"] == 2 and empty["i_peak"] == 0.0


def test_eq35_read_backwards_reproduces_the_papers_printed_estimate():
    """peak at v/v_fs = 1.32, relative curvature about -110 => beta = 10.5 and tau0 = 28.79."""
    import os
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_printed_values.txt")):
        if line.strip() and not line.startswith("#"):
            name, val, tol = line.split()[:3]
            gold[name] = (float(val), float(tol))
    beta, tau0 = peak.ejecta_from_peak(1.32, -110.0)
    assert beta == pytest.approx(gold["eq35_beta_from_curvature"][0], abs=gold["eq35_beta_from_curvature"][1])
    _, tau0_rounded = peak.ejecta_from_peak(1.32, -(10.5 ** 2))            # the paper continues with the rounded beta
    assert tau0_rounded == pytest.approx(gold["eq35_tau0_from_position"][0], abs=gold["eq35_tau0_from_position"][1])
    assert tau0 == pytest.approx(28.79, rel=5e-3)
    assert peak.ejecta_from_peak(1.2, 0.0) == (0.0, 0.0) and peak.ejecta_from_peak(1.2, 3.0) == (0.0, 0.0)
    r = peak.spectrum_peak(np.maximum(3.0 - 40.0 * (np.arange(512) / 512 * 3 + 3 / 1024 - 1.3) ** 2, 0), 1, 0.0, 6000.0, 2000.0)
    assert r["beta_eq35"] == pytest.approx(math.sqrt(-r["curvature"])) and r["tau0_eq35"] == pytest.approx(
        math.exp(r["beta_eq35"] * (r["x_peak"] - 1.0)))

