"""Pins for the MULTI-CLASS branch of the oracle Monte-Carlo (pick_class, the per-class phase-table offset and the per-class
albedo in oracle/pdv_oracle_mc.c::run_history) -- CPU only.  Pin P18 of DESIGN.md section 1.

Every 16-class result (configs 3 and 5, the parameter sweeps of row f1) rests on that branch.  The expected values here are
closed forms and quadratures written out in this file (Eq. 8: a particle of class c is hit with probability
P_c ~ w_c d_c^2 K_ext,c; Eq. 11: it scatters with probability omega0_c = K_sca,c / K_ext,c; Eq. 13:
the scattering angle follows the phase function of THAT class), never a second call of the oracle's own
formula.  Each of the three one-line mistakes
    xi >= p_cum[c]  ->  xi >= p_cum[c+1]      (pick_class)
    phase + c (K+1) ->  phase                 (table of class 0 for every class)
    omega0[c]       ->  omega0[0]             (albedo of class 0 for every class)
turns at least one test of this file red (checked by editing a copy of the C file).
"""
import dataclasses
import math

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud, mc

from histcmp import compare, compare_to_expectation

MU_A = 1.0 - W.APERTURE_SR / (2.0 * math.pi)


def _run_opts(n, **kw):
    o = dict(W.config(1)["run"])
    o.update(n_photons=int(n), seed=4242)
    o.update(kw)
    return o


def _T_of_v(c, v):
    """Closed form: vertical optical depth above velocity v for Eq. 20 truncated to [v_fs, v_max]."""
    E = math.exp(-c.beta * (c.v_max / c.v_fs - 1.0))
    return c.tau_ext * (np.exp(-c.beta * (np.asarray(v) / c.v_fs - 1.0)) - E) / (1.0 - E)


def _hand_made(base, p_class, omega0, cosines):
    """`base` (one class) turned into a cloud of len(p_class) classes whose phase functions are deltas: class c always
    scatters by cos(theta) = cosines[c].  Depth table, tau_ext and velocities are those of `base`."""
    K = base.phase.shape[1] - 1
    n = len(p_class)
    return dataclasses.replace(
        base, diameters=np.full(n, base.diameters[0]), number_weights=np.full(n, 1.0 / n),
        k_ext=np.full(n, base.k_ext[0]), k_sca=np.asarray(omega0) * base.k_ext[0], g=np.asarray(cosines, dtype=float),
        omega0=np.asarray(omega0, dtype=float), p_class=np.asarray(p_class, dtype=float),
        phase=np.repeat(np.asarray(cosines, dtype=float)[:, None], K + 1, axis=1), surface_reflectivity=0.0)


# ---------------------------------------------------------------------------------------------------------------------------
def test_delta_classes_closed_form_per_class_P18(cfg2_oracle_cloud):
    """Four classes with delta phase functions at four different angles, four different albedos, four different hit
    probabilities; single-scatter-only, R = 0, aperture 2 pi.  The launch direction is (0,0,-1), so after ONE scatter of
    class c the photon travels with mu = -cos(theta_c) exactly (Eq. 17), and a photon that leaves the top after exactly one
    particle event tells its class by its exit cosine.  For a class that sends the photon up (mu_c > 0):
        first event at depth T (density e^-T on [0, tau]) x class c (P_c) x escape without a second event (e^{-T/mu_c})
        => N_c ~ Binomial(N, P_c (1 - e^{-a tau}) / a),  a = 1 + 1/mu_c,   every such history carries weight omega0_c exactly.
    A class that sends it further down (mu_f < 0) reaches the surface with probability e^{-(tau-T)/|mu_f|}:
        absorbed_surface / N = e^-tau + P_f omega0_f (e^-tau - e^{-b tau}) / (b - 1),  b = 1/|mu_f|    (R = 0).
    First-collision capture (implicit, Eq. 11):  absorbed_particles / N = (1 - e^-tau) sum_c P_c (1 - omega0_c)."""
    p = np.array([0.10, 0.40, 0.20, 0.30])
    om = np.array([0.90, 0.35, 0.60, 0.75])
    ct = np.array([-1.0, -0.5, -0.25, 0.5])               # classes 0-2 send the photon up, class 3 down with mu = -0.5
    c = _hand_made(cfg2_oracle_cloud, p, om, ct)
    tau = c.tau_ext
    n = 2_000_000
    r = mc.run(c, _run_opts(n, single_scatter_only=1, aperture_sr=2.0 * math.pi), trace=True)
    tr = r.trace
    once = tr[(tr["n_scatter"] == 1) & (tr["n_reflect"] == 0) & (tr["fate"] == 0)]
    seen = 0
    for k in range(3):
        mu_c = -ct[k]
        sel = once[np.abs(once["mu_exit"] - mu_c) < 1e-12]
        a = 1.0 + 1.0 / mu_c
        prob = p[k] * (1.0 - math.exp(-a * tau)) / a
        assert abs(len(sel) - n * prob) < 5.0 * math.sqrt(n * prob * (1.0 - prob)), (k, len(sel), n * prob)
        assert len(sel) > 10_000 and np.all(sel["w"] == om[k])           # the albedo of THAT class, to the last bit
        # Doppler shift of one event at velocity v: (mu_out - mu_in) v / 2 with mu_in = -1 (Eq. 4)
        assert sel["vt"].min() >= 0.5 * (1.0 + mu_c) * c.v_fs - 1e-9 and sel["vt"].max() <= 0.5 * (1.0 + mu_c) * c.v_max + 1e-9
        seen += len(sel)
    assert seen == len(once)                                             # no other exit cosine exists after one scatter
    b = 1.0 / 0.5
    e_surf = math.exp(-tau) + p[3] * om[3] * (math.exp(-tau) - math.exp(-b * tau)) / (b - 1.0)
    assert r.stats["absorbed_surface"] == pytest.approx(n * e_surf, abs=5.0 * math.sqrt(n * e_surf))
    first = 1.0 - math.exp(-tau)
    e_abs = first * float(np.sum(p * (1.0 - om)))
    var_abs = first * float(np.sum(p * (1.0 - om) ** 2)) - e_abs ** 2
    assert r.stats["absorbed_particles"] == pytest.approx(n * e_abs, abs=5.0 * math.sqrt(n * var_abs))
    assert abs(r.conservation_residual()) < 1e-10 * n


def test_two_class_backscatter_histogram_scales_with_P0_omega0_P18(cfg2_oracle_cloud):
    """Class 0 a delta at theta = pi, class 1 a delta at theta = 0 (the photon flies on, to a second event or to the black
    surface): the single-backscatter histogram of pin P2 scaled by exactly P_0 omega0_0,
        H_k / N = P_0 omega0_0 / 2 [exp(-2 T(v_{k+1})) - exp(-2 T(v_k))]           (Eq. 8, 11)."""
    p, om = np.array([0.35, 0.65]), np.array([0.80, 0.50])
    c = _hand_made(cfg2_oracle_cloud, p, om, [-1.0, 1.0])
    n = 2_000_000
    r = mc.run(c, _run_opts(n, single_scatter_only=1, aperture_sr=1e-3))
    edges = np.linspace(0.0, 6000.0, 513)
    Tk = _T_of_v(c, np.clip(edges, c.v_fs, c.v_max))
    expected = 0.5 * p[0] * om[0] * (np.exp(-2 * Tk[1:]) - np.exp(-2 * Tk[:-1]))
    res = compare_to_expectation(r.hist, r.hist2, n, expected)
    assert res["worst"] < 5.0 and res["ndf"] > 100
    var = n * expected.sum() * om[0]                                     # Poisson count of weights omega0_0
    assert r.stats["detected"] == pytest.approx(n * expected.sum(), abs=5.0 * math.sqrt(var))
    # swapping the two classes (same tables, same albedos, other probabilities) scales it by P_1 omega0_1 instead
    c2 = _hand_made(cfg2_oracle_cloud, p, om, [1.0, -1.0])
    r2 = mc.run(c2, _run_opts(n, single_scatter_only=1, aperture_sr=1e-3))
    e2 = expected * (p[1] * om[1]) / (p[0] * om[0])
    assert compare_to_expectation(r2.hist, r2.hist2, n, e2)["worst"] < 5.0
    assert r2.stats["detected"] == pytest.approx(n * e2.sum(), abs=5.0 * math.sqrt(n * e2.sum() * om[1]))


@pytest.fixture(scope="module")
def three_mie_classes():
    """Tin spheres of 0.15, 0.4 and 5 um (albedo 0.25 / 0.84 / 0.93, g -0.14 / -0.17 / +0.54), number weights chosen so
    that all three are hit often."""
    params = dict(W._cloud(2.0, 4.0, 2000.0, diameter_um=5.0), diameters=[0.15e-6, 0.4e-6, 5.0e-6],
                  number_weights=[20000.0, 200.0, 1.0])
    c = cloud.build_cloud(params)
    assert c.omega0[0] < 0.3 < 0.8 < c.omega0[1] < 0.9 < c.omega0[2] and c.g[0] < -0.1 and c.g[2] > 0.5
    assert np.all(c.p_class > 0.15)
    return c


def test_single_scatter_quadrature_summed_over_mie_classes_P8_P18(three_mie_classes):
    """SURVEY.md 8(c) pin P8 as it is written, with the sum over classes:
        H_k/N = sum_c P_c omega0_c int dT e^-T int_{mu_a}^1 dmu p~_c(-mu) e^{-T/mu} 1[(1+mu) v(T)/2 in bin k]
    (midpoint rule in (v, mu); p~_c = piecewise-constant density of D_K of class c in cos(theta)); plus the first-collision
    capture  absorbed_particles / N = (1 - e^-tau) sum_c P_c (1 - omega0_c)  with R = 0."""
    c = dataclasses.replace(three_mie_classes, surface_reflectivity=0.0)
    n = 4_000_000
    r = mc.run(c, _run_opts(n, single_scatter_only=1))
    n_v, n_mu = 16000, 500
    v = c.v_fs + (np.arange(n_v) + 0.5) / n_v * (c.v_max - c.v_fs)
    E = math.exp(-c.beta * (c.v_max / c.v_fs - 1.0))
    dT = c.tau_ext * (c.beta / c.v_fs) * np.exp(-c.beta * (v / c.v_fs - 1.0)) / (1.0 - E) * (c.v_max - c.v_fs) / n_v
    T = _T_of_v(c, v)
    mu = MU_A + (np.arange(n_mu) + 0.5) / n_mu * (1.0 - MU_A)
    dens = np.zeros(n_mu)
    per_class = []
    for k in range(c.n_classes):
        M = c.phase[k]
        K = M.size - 1
        cell = np.clip(np.searchsorted(M, -mu, side="right") - 1, 0, K - 1)
        d_k = 1.0 / (K * (M[cell + 1] - M[cell]))                         # density of cos(theta) = -mu under D_K of class k
        per_class.append(float(c.p_class[k] * c.omega0[k] * d_k.mean()))
        dens += c.p_class[k] * c.omega0[k] * d_k
    # the three classes contribute comparably, so that a wrong class weight, table or albedo moves the sum by tens of percent
    assert min(per_class) > 0.1 * max(per_class)
    wgt = (dT * np.exp(-T))[:, None] * np.exp(-T[:, None] / mu[None, :]) * (dens * (1 - MU_A) / n_mu)[None, :]
    vt = 0.5 * (1.0 + mu)[None, :] * v[:, None]
    expected, _ = np.histogram(vt.ravel(), bins=512, range=(0.0, 6000.0), weights=wgt.ravel())
    res = compare_to_expectation(r.hist, r.hist2, n, expected, min_eff=50.0)
    assert res["worst"] < 5.0 and res["ndf"] >= 20
    tot = expected.sum()
    assert r.stats["detected"] == pytest.approx(n * tot, abs=5.0 * math.sqrt(n * tot))
    first = 1.0 - math.exp(-c.tau_ext)
    e_abs = first * float(np.sum(c.p_class * (1.0 - c.omega0)))
    var_abs = first * float(np.sum(c.p_class * (1.0 - c.omega0) ** 2)) - e_abs ** 2
    assert r.stats["absorbed_particles"] == pytest.approx(n * e_abs, abs=5.0 * math.sqrt(n * var_abs))


def test_analog_capture_agrees_with_implicit_on_mie_classes_P18(three_mie_classes):
    """Eq. 11 literally (absorbed with probability 1 - omega0_c) against implicit capture (weight omega0_c): the analog branch
    reads omega0[c] at a different place of run_history."""
    c = three_mie_classes
    n = 2_000_000
    a = mc.run(c, _run_opts(n, seed=11))
    b = mc.run(c, _run_opts(n, seed=12, mode=1))
    res = compare(a.hist, a.hist2, n, b.hist, b.hist2, n)
    assert res["worst"] < 5.0 and res["ndf"] > 50
    sa, sb = a.stats["absorbed_particles"] / n, b.stats["absorbed_particles"] / n
    assert sa == pytest.approx(sb, abs=5.0 * math.sqrt(2.0 * sb / n))
    # analog first collision: the absorbed COUNT after one event, in closed form
    e1 = mc.run(dataclasses.replace(c, surface_reflectivity=0.0), _run_opts(n, seed=13, mode=1, single_scatter_only=1))
    prob = (1.0 - math.exp(-c.tau_ext)) * float(np.sum(c.p_class * (1.0 - c.omega0)))
    assert e1.stats["absorbed_particles"] == pytest.approx(n * prob, abs=5.0 * math.sqrt(n * prob * (1 - prob)))


@pytest.mark.parametrize("which,mode", [("three_mie", 0), ("three_mie", 1), ("config3", 0)])
def test_shared_philox_stream_on_a_polydisperse_cloud_P18(three_mie_classes, which, mode):
    """rng_mode 1 with several classes (D2: two Philox blocks feed three flights, class words from W2, W5 and their
    low bytes) is statistically the same process as the independent generator: on three Mie classes that differ strongly
    (a class word that lost a bit, or one flight of three reading another word, changes which class is hit and with it the
    albedo and the angular law), and on the 16-class cloud of config 3."""
    c = three_mie_classes if which == "three_mie" else cloud.build_cloud(W.config(2)["clouds"][0])
    n = 1_500_000
    a = mc.run(c, _run_opts(n, seed=101, mode=mode))
    b = mc.run(c, _run_opts(n, seed=202, mode=mode), rng_mode=1)      # mode 1 also reads the absorption words of the companion blocks
    res = compare(a.hist, a.hist2, n, b.hist, b.hist2, n)
    assert res["worst"] < 5.0 and res["ndf"] > 50
    assert res["chi2"] < res["ndf"] + 5 * math.sqrt(2 * res["ndf"])
    for key, sd in (("particle_events", 25.0), ("surface_reflections", 1.0)):
        assert a.stats[key] / n == pytest.approx(b.stats[key] / n, abs=5.0 * sd * math.sqrt(2.0 / n))
    for key in ("detected", "escaped", "absorbed_particles", "absorbed_surface"):
        assert a.stats[key] / n == pytest.approx(b.stats[key] / n, abs=5.0 * math.sqrt(2.0 / n))
