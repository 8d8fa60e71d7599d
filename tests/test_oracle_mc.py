"""Pins for the oracle Monte-Carlo (oracle/pdv_oracle_mc.c through oracle/mc.py) -- CPU only.

SURVEY.md 8(c) pins P1 (Beer-Lambert), P2 (exact 2v/lambda shift, closed-form histogram), P3 (Eq. 4 vs
sign-corrected Eq. 18), P6 (rotation Eq. 16/17), P8 (single-scatter integral by quadrature, Eq. 28/31
limit), P9 (surface model), P11 (weight conservation), P12 (estimator equivalences) and the
published Philox4x32-10 known-answer vectors.  Expected values are closed forms / quadratures written
out here, never a second call of the oracle's own formula.
"""
import dataclasses
import math
import os

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud, mc

from histcmp import compare, compare_to_expectation

MU_A = 1.0 - W.APERTURE_SR / (2.0 * math.pi)


def _T_of_v(c, v):
    """Closed form: vertical optical depth above velocity v for Eq. 20 truncated to [v_fs, v_max]."""
    E = math.exp(-c.beta * (c.v_max / c.v_fs - 1.0))
    return c.tau_ext * (np.exp(-c.beta * (np.asarray(v) / c.v_fs - 1.0)) - E) / (1.0 - E)


def _run_opts(n, **kw):
    o = dict(W.config(1)["run"])
    o.update(n_photons=int(n), seed=12345)
    o.update(kw)
    return o


# ------------------------------------------------------------------------------------------ Philox
def test_philox4x32_10_known_answers():
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        words = [int(t, 16) for t in line.split()]
        assert mc.philox4x32_10(words[0:4], words[4:6]) == words[6:10]
        n += 1
    assert n == 3


# ------------------------------------------------------------------------------------------ P6
def test_rotation_preserves_norm_and_angle_P6():
    rng = np.random.default_rng(1)
    for _ in range(300):
        u = rng.normal(size=3)
        u /= np.linalg.norm(u)
        ct, phi = rng.uniform(-1, 1), rng.uniform(0, 2 * math.pi)
        v = mc.rotate(u, ct, phi)
        assert np.linalg.norm(v) == pytest.approx(1.0, abs=1e-12)
        assert float(v @ u) == pytest.approx(ct, abs=1e-12)
    # pole case, Eq. 17: u = (0,0,-1) and theta -> u_z' = -cos(theta)
    for ct in (-1.0, -0.3, 0.7, 1.0):
        v = mc.rotate([0.0, 0.0, -1.0], ct, 0.4)
        assert v[2] == pytest.approx(-ct, abs=1e-15) and np.linalg.norm(v) == pytest.approx(1.0, abs=1e-15)
    # z row of Eq. 16 as printed: u_z' = -sin(th) cos(phi) sqrt(1-u_z^2) + u_z cos(th)
    u = np.array([0.36, 0.48, 0.8])
    ct, phi = 0.3, 1.1
    assert mc.rotate(u, ct, phi)[2] == pytest.approx(-math.sqrt(1 - ct * ct) * math.cos(phi) * 0.6 + 0.8 * ct, abs=1e-14)
    # azimuthal symmetry: averaging over a uniform phi grid leaves cos(theta) u
    acc = sum(mc.rotate(u, ct, 2 * math.pi * i / 64) for i in range(64)) / 64
    assert np.allclose(acc, ct * u, atol=1e-13)


def test_mean_cosine_after_n_scatterings_is_g_to_the_n_P6(cfg2_oracle_cloud):
    """Infinite medium: <u_n . u_0> = g^n for any phase function with mean cosine g."""
    c = cfg2_oracle_cloud
    rng = np.random.default_rng(7)
    M, K = c.phase[0], c.phase.shape[1] - 1
    n_s, n = 3, 12000
    acc = 0.0
    for _ in range(n):
        u = np.array([0.0, 0.6, -0.8])
        for _ in range(n_s):
            t = rng.random() * K
            k = int(t)
            u = mc.rotate(u, M[k] + (M[k + 1] - M[k]) * (t - k), 2 * math.pi * rng.random())
        acc += u[1] * 0.6 - u[2] * 0.8
    g = float(c.g[0])
    assert acc / n == pytest.approx(g**n_s, abs=5 * 0.6 / math.sqrt(n))


# ------------------------------------------------------------------------------------------ P1 / P9
def test_beer_lambert_pure_absorber_P1(cfg2_oracle_cloud):
    """omega0 = 0, analog: photons reaching the surface ~ Binomial(N, exp(-tau_ext)) (Eq. 7/10), and the
    detected ones are exactly the direct-reflection term  N e^-tau R int_{mu_a}^1 q(mu) e^{-tau/mu} dmu,
    q(mu) = (2/pi)/sqrt(1-mu^2)  (theta uniform)."""
    c = dataclasses.replace(cfg2_oracle_cloud, omega0=np.zeros(1))
    n = 2_000_000
    r = mc.run(c, _run_opts(n, mode=1))
    reached = r.stats["absorbed_surface"] + r.stats["surface_reflections"]
    p = math.exp(-c.tau_ext)
    assert abs(reached - n * p) < 4.5 * math.sqrt(n * p * (1 - p))
    th = (np.arange(20000) + 0.5) / 20000 * math.acos(MU_A)
    p_det = p * c.surface_reflectivity * (2 / math.pi) * np.sum(np.exp(-c.tau_ext / np.cos(th))) * (th[1] - th[0])
    det = r.stats["detected"]
    assert abs(det - n * p_det) < 4.5 * math.sqrt(n * p_det)
    # every detected photon was shifted by (mu_out + 1) v_fs / 2 in [0.992, 1] v_fs  (Eq. 4, one event at v_fs)
    dv = 6000.0 / 512
    k_lo, k_hi = int(0.5 * (1 + MU_A) * c.v_fs / dv), int(c.v_fs / dv)
    assert r.hist[k_lo:k_hi + 1].sum() == pytest.approx(det, abs=1e-9) and r.stats["particle_events"] > 0


@pytest.mark.parametrize("surface_model,mean_mu,frac", [(0, 2 / math.pi, math.acos(MU_A) / (math.pi / 2)),
                                                         (1, 2.0 / 3.0, 1 - MU_A**2)])
def test_surface_reflection_law_P9(cfg2_oracle_cloud, surface_model, mean_mu, frac):
    """Empty cloud (tau -> 0), R = 1: every photon reflects once; paper model: theta uniform => <mu> = 2/pi and
    P(inside 0.1 sr) = acos(mu_a)/(pi/2) = 0.1137; Lambertian: <mu> = 2/3, P = 1 - mu_a^2."""
    c = dataclasses.replace(cfg2_oracle_cloud, tau_ext=1e-9, T_edge=cfg2_oracle_cloud.T_edge * 1e-9 / cfg2_oracle_cloud.tau_ext,
                            surface_reflectivity=1.0, surface_model=surface_model)
    n = 400_000
    r = mc.run(c, _run_opts(n), trace=True)
    tr = r.trace
    assert np.all(tr["n_reflect"] == 1) and np.all(tr["n_scatter"] == 0)
    assert tr["mu_exit"].mean() == pytest.approx(mean_mu, abs=5 * 0.31 / math.sqrt(n))
    assert (tr["fate"] == 0).mean() == pytest.approx(frac, abs=5 * math.sqrt(frac / n))
    assert np.allclose(tr["vt"], 0.5 * (tr["mu_exit"] + 1.0) * c.v_fs, rtol=1e-14)
    if surface_model == 0:
        assert frac == pytest.approx(0.1137, abs=1e-4)


# ------------------------------------------------------------------------------------------ P2 / P3
def test_single_backscatter_shift_is_2v_over_lambda_P2(cfg2_oracle_cloud):
    """Phase function = delta at theta = pi, single-scatter mode, R = 0: every tallied photon carries v~ = v of
    its scatterer (Eq. 4: (n_s - n).v w_r/c = 2 v w_r/c) and the histogram has the closed form
    H_k/N = omega0/2 [exp(-2 T(v_k+1)) - exp(-2 T(v_k))]."""
    c0 = cfg2_oracle_cloud
    K = c0.phase.shape[1] - 1
    c = dataclasses.replace(c0, phase=-np.ones((1, K + 1)), surface_reflectivity=0.0)
    n = 1_000_000
    r = mc.run(c, _run_opts(n, single_scatter_only=1, aperture_sr=1e-3), trace=True)
    tr = r.trace
    det = tr[(tr["fate"] == 0) & (tr["w"] > 0)]          # R = 0: photons that met the surface carry weight 0
    assert len(det) > 1000 and np.all(det["n_scatter"] == 1) and np.all(det["mu_exit"] == 1.0)
    assert det["vt"].min() >= c.v_fs - 1e-9 and det["vt"].max() <= c.v_max + 1e-9
    edges = np.linspace(0.0, 6000.0, 513)
    Tk = _T_of_v(c, np.clip(edges, c.v_fs, c.v_max))
    expected = 0.5 * float(c.omega0[0]) * (np.exp(-2 * Tk[1:]) - np.exp(-2 * Tk[:-1]))
    res = compare_to_expectation(r.hist, r.hist2, n, expected)
    assert res["worst"] < 5.0 and res["ndf"] > 100
    assert r.stats["detected"] == pytest.approx(n * expected.sum(), abs=5 * math.sqrt(n * expected.sum()))


def test_single_scatter_peak_position_Eq31():
    """Thick cloud, all-backward single scattering: spectrum ~ f(v) exp(-2 T(v)) peaks at
    v/v_fs = 1 + ln(2 tau_ext)/beta  (Eq. 28/31 with tau0 <-> 2 tau_ext, reading on P8)."""
    params = W._cloud(5.0, 4.0, 2000.0, diameter_um=5.0)
    K = params["n_phase_bins"]
    c = cloud.build_cloud(params, phase_override=-np.ones((1, K + 1)))
    n = 3_000_000
    r = mc.run(c, _run_opts(n, single_scatter_only=1, aperture_sr=1e-3))
    sm = np.convolve(r.hist, np.ones(9) / 9, mode="same")
    v_peak = (np.argmax(sm) + 0.5) * 6000.0 / 512
    # E (truncation at 3 v_fs) shifts the exponential law by a constant: the peak condition is unchanged
    expected = c.v_fs * (1.0 + math.log(2.0 * c.tau_ext / (1.0 - math.exp(-8.0))) / c.beta)
    assert v_peak == pytest.approx(expected, abs=3 * 6000.0 / 512)


def test_per_event_equals_per_leg_doppler_P3(cfg2_oracle_cloud):
    """Eq. 4 summed per event == Eq. 18 with the sign fixed, summed per flight leg (source, detector at rest)."""
    r = mc.run(cfg2_oracle_cloud, _run_opts(200_000), trace=True)
    tr = r.trace
    out = tr[(tr["fate"] == 0) | (tr["fate"] == 1)]
    assert len(out) > 50_000
    assert np.max(np.abs(out["vt"] - out["vt_leg"])) < 1e-8
    assert out["n_scatter"].max() > 20


# ------------------------------------------------------------------------------------------ P8
def test_single_scatter_mode_matches_quadrature_P8(cfg2_oracle_cloud):
    """Single-scatter-only, R = 0:  H_k/N = omega0 int dT e^-T int_{mu_a}^1 dmu p~(-mu) e^{-T/mu} 1[(1+mu) v(T)/2 in bin k]
    by a midpoint rule in (v, mu); p~ = piecewise-constant density of D_K in cos(theta)."""
    c = dataclasses.replace(cfg2_oracle_cloud, surface_reflectivity=0.0)
    n = 4_000_000
    r = mc.run(c, _run_opts(n, single_scatter_only=1))
    M = c.phase[0]
    K = M.size - 1
    n_v, n_mu = 16000, 500
    v = c.v_fs + (np.arange(n_v) + 0.5) / n_v * (c.v_max - c.v_fs)
    E = math.exp(-c.beta * (c.v_max / c.v_fs - 1.0))
    dT = c.tau_ext * (c.beta / c.v_fs) * np.exp(-c.beta * (v / c.v_fs - 1.0)) / (1.0 - E) * (c.v_max - c.v_fs) / n_v
    T = _T_of_v(c, v)
    mu = MU_A + (np.arange(n_mu) + 0.5) / n_mu * (1.0 - MU_A)
    kcell = np.clip(np.searchsorted(M, -mu, side="right") - 1, 0, K - 1)
    dens = 1.0 / (K * (M[kcell + 1] - M[kcell]))                      # density of cos(theta) = -mu
    wgt = float(c.omega0[0]) * (dT * np.exp(-T))[:, None] * np.exp(-T[:, None] / mu[None, :]) * (dens * (1 - MU_A) / n_mu)[None, :]
    vt = 0.5 * (1.0 + mu)[None, :] * v[:, None]
    expected, _ = np.histogram(vt.ravel(), bins=512, range=(0.0, 6000.0), weights=wgt.ravel())
    res = compare_to_expectation(r.hist, r.hist2, n, expected, min_eff=50.0)
    assert res["worst"] < 5.0 and res["ndf"] >= 20
    tot = expected.sum()
    assert r.stats["detected"] == pytest.approx(n * tot, abs=5 * math.sqrt(n * tot))
    assert r.stats["truncated"] > 0.1 * n


# ------------------------------------------------------------------------------------------ P11
@pytest.mark.parametrize("kw", [dict(), dict(mode=1), dict(max_events=5, roulette_survival=0.3),
                                dict(single_scatter_only=1), dict(mode=1, max_events=3, roulette_survival=0.5)])
def test_weight_conservation_P11(cfg2_oracle_cloud, kw):
    n = 300_000
    r = mc.run(cfg2_oracle_cloud, _run_opts(n, **kw))
    assert abs(r.conservation_residual()) < 1e-10 * n
    assert r.stats["histories"] == n
    assert r.hist.sum() == pytest.approx(r.stats["detected"], rel=1e-12)


# ------------------------------------------------------------------------------------------ P12
def _pair(c, n, kw_a, kw_b, run_a=None, run_b=None):
    a = mc.run(c, _run_opts(n, seed=101, **kw_a), **(run_a or {}))
    b = mc.run(c, _run_opts(n, seed=202, **kw_b), **(run_b or {}))
    res = compare(a.hist, a.hist2, n, b.hist, b.hist2, n)
    return a, b, res


def test_analog_vs_implicit_capture_P12(cfg2_oracle_cloud):
    a, b, res = _pair(cfg2_oracle_cloud, 1_500_000, dict(mode=0), dict(mode=1))
    assert res["worst"] < 5.0 and res["ndf"] > 50
    assert res["chi2"] < res["ndf"] + 5 * math.sqrt(2 * res["ndf"])


def test_roulette_is_unbiased_P12(cfg2_oracle_cloud):
    """Survival 0.8 from event 6 on keeps the weight variance finite (omega0^2/p < 1 per step), so the 5 sigma rule
    applies; a harsh roulette (p = 0.25 at every event) has a heavy-tailed weight law and is no test of bias."""
    a, b, res = _pair(cfg2_oracle_cloud, 1_500_000, dict(), dict(max_events=6, roulette_survival=0.8))
    assert b.stats["roulette_killed"] > 0 and res["worst"] < 5.0
    assert res["chi2"] < res["ndf"] + 5 * math.sqrt(2 * res["ndf"])


def test_depth_table_vs_analytic_profile_P12(cfg2_oracle_cloud):
    a, b, res = _pair(cfg2_oracle_cloud, 1_500_000, dict(), dict(), run_b=dict(analytic_profile=True))
    assert res["worst"] < 5.0
    assert res["chi2"] < res["ndf"] + 5 * math.sqrt(2 * res["ndf"])


def test_table_vs_exact_mie_rejection_P12(cfg2_oracle_cloud):
    """D_1024 against the paper's own acceptance-rejection on the exact Mie function."""
    a, b, res = _pair(cfg2_oracle_cloud, 600_000, dict(), dict(),
                      run_b=dict(exact_mie=dict(m=complex(W.M_RE, W.M_IM), wavelength=W.WAVELENGTH)))
    assert res["worst"] < 5.0
    assert res["chi2"] < res["ndf"] + 5 * math.sqrt(2 * res["ndf"])
    assert b.stats["particle_events"] / 600_000 == pytest.approx(a.stats["particle_events"] / 600_000, rel=0.01)


def test_shared_philox_stream_agrees_with_independent_generator(cfg2_oracle_cloud):
    """rng_mode 1 (the counter-based stream both sides implement, D1/D2) is statistically the same process."""
    a, b, res = _pair(cfg2_oracle_cloud, 1_500_000, dict(), dict(), run_b=dict(rng_mode=1))
    assert res["worst"] < 5.0
    assert res["chi2"] < res["ndf"] + 5 * math.sqrt(2 * res["ndf"])


def test_thread_count_and_id_ranges_do_not_change_results(cfg2_oracle_cloud):
    """Histories are keyed by photon id: [0,n) on 1 thread == [0,n/2) + [n/2,n) on 3 threads (up to summation order)."""
    n = 60_000
    for rng_mode in (0, 1):
        a = mc.run(cfg2_oracle_cloud, _run_opts(n), n_threads=1, rng_mode=rng_mode)
        b1 = mc.run(cfg2_oracle_cloud, _run_opts(n), n_photons=n // 2, first_id=0, n_threads=3, rng_mode=rng_mode)
        b2 = mc.run(cfg2_oracle_cloud, _run_opts(n), n_photons=n // 2, first_id=n // 2, n_threads=3, rng_mode=rng_mode)
        assert np.allclose(a.hist, b1.hist + b2.hist, rtol=0, atol=1e-9)
        assert a.stats["particle_events"] == b1.stats["particle_events"] + b2.stats["particle_events"]


@pytest.mark.parametrize("m0,d_um", [(1.0, 5.0), (3.0, 2.0)])
def test_multiple_scattering_core_obeys_the_mean_path_invariance(m0, d_um):
    """The multiple-scattering transport itself, pinned by a theorem instead of a closed form: in a NON-ABSORBING medium
    under uniform diffuse (Lambertian) illumination the mean path length of a photon inside is 4 V / S, whatever the
    phase function and the optical thickness (the mean-chord-length invariance; equilibrium radiance is uniform and
    isotropic).  For the slab in optical units V/S = tau_ext per unit of open surface, with a Lambertian, lossless
    bottom, so per history:
        <optical path> = <particle events> = 4 tau_ext,   <surface reflections> = 1   (bottom area = open area),
    and what leaves is Lambertian again: P(mu_exit >= mu_a) = 1 - mu_a^2, <mu_exit> = 2/3.
    Cloud: real refractive index 1.5 (K_abs = 0, albedo 1) with the full Mie phase table, Lambertian surface, R = 1.
    A wrong sign or factor in T' = T - mu s, in the z row of Eq. 16 or in the reflection law breaks every one of these."""
    params = dict(W._cloud(m0, 4.0, 2000.0, diameter_um=d_um), m_re=1.5, m_im=0.0, surface_model=1,
                  surface_reflectivity=1.0)
    c = cloud.build_cloud(params)
    assert np.allclose(c.omega0, 1.0, atol=1e-12)
    n = 400_000
    run = dict(W.config(1)["run"], aperture_sr=0.1, v_lo=-20000.0, v_hi=20000.0)
    r = mc.run(c, dict(run, seed=31), n_photons=n, launch_model=1, trace=True)
    ev = r.trace["n_scatter"].astype(np.float64)
    assert r.stats["particle_events"] / n == pytest.approx(4.0 * c.tau_ext, abs=5 * ev.std() / math.sqrt(n))
    rf = r.trace["n_reflect"].astype(np.float64)
    assert r.stats["surface_reflections"] / n == pytest.approx(1.0, abs=5 * rf.std() / math.sqrt(n))
    mu_a = mc.aperture_mu(0.1)
    p_in = 1.0 - mu_a ** 2
    assert (r.stats["detected"] + r.stats["underflow"] + r.stats["overflow"]) / n == pytest.approx(
        p_in, abs=5 * math.sqrt(p_in / n))
    assert float(np.mean(r.trace["mu_exit"])) == pytest.approx(2.0 / 3.0, abs=5 * math.sqrt(1.0 / 18.0 / n))
    # the same cloud under the paper's collimated beam does NOT have these values: the pin is not vacuous
    r0 = mc.run(c, dict(run, seed=31), n_photons=100_000)
    assert abs(r0.stats["particle_events"] / 100_000 - 4.0 * c.tau_ext) > 0.05 * 4.0 * c.tau_ext


@pytest.mark.parametrize("kw", [dict(), dict(mode=1)])
def test_rigid_cloud_doppler_telescopes_to_the_exit_angle_P17(kw):
    """A closed form for the MULTIPLE-scattering spectrum, in a special cloud: if every particle and the free surface move
    with the same velocity v, the shifts of Eq. 4 telescope over any number of events,
        v~ = 1/2 sum_k (mu_k_out - mu_k_in) v = 1/2 (mu_exit - mu_launch) v = 1/2 (1 + mu_exit) v     (collimated launch),
    so every detected photon (mu_exit >= mu_a) lands in [ (1 + mu_a)/2 v, v ] whatever happened to it on the way -- with
    0.1 sr and v = 2000 m/s that is [1984.08, 2000] m/s out of a 0-6000 m/s axis.  A dropped, doubled or wrongly signed
    term at ANY event of a long history puts weight outside.  Cloud: tabulated profile with all the mass within 2 mm/s of
    v_fs, 2 mg/cm^2 (7 events per history on average, up to ~70)."""
    base = W.config(1)["clouds"][0]
    params = dict(base, profile_kind=1, prof_v=np.array([2000.0, 2000.002]), prof_cum_mass=np.array([0.0, 1.0]),
                  vmax_ratio=1.000001)
    c = cloud.build_cloud(params)
    assert c.v_max == pytest.approx(2000.002, abs=1e-9)
    n, nb, lo, hi = 400_000, 8000, 1900.0, 2100.0
    run = dict(W.config(1)["run"], n_bins=nb, v_lo=lo, v_hi=hi, **kw)
    r = mc.run(c, dict(run, seed=17), n_photons=n, trace=True)
    assert r.stats["particle_events"] / n > 3.5 and r.trace["n_scatter"].max() > 30      # analog histories are shorter
    assert r.stats["underflow"] == 0.0 and r.stats["overflow"] == 0.0
    mu_a = mc.aperture_mu(0.1)
    centres = lo + (np.arange(nb) + 0.5) * (hi - lo) / nb
    inside = (centres > 0.5 * (1 + mu_a) * 2000.0 - 0.05) & (centres < 2000.002 + 0.05)
    assert r.hist[~inside].sum() == 0.0 and r.hist[inside].sum() == pytest.approx(r.stats["detected"], rel=1e-12)
    assert r.stats["detected"] / n > 0.01
    # history by history: v~ = (1 + mu_exit) v / 2 for every photon that left through the top, detected or not
    out = r.trace["fate"] <= 1
    assert np.max(np.abs(r.trace["vt"][out] - 0.5 * (1.0 + r.trace["mu_exit"][out]) * 2000.0)) < 0.002 * 40


# ------------------------------------------------------------------------------------------ P20
def _double_scatter_quadrature(c, omega0, mu_a, n1=240, nm=120, ns=96, n2=12):
    """Detected weight per launched photon of the histories that scatter EXACTLY twice (no reflection) in a cloud with an
    isotropic phase function, as nodes (v~, weight) of a Gauss-Legendre rule over (T1, mu1, s, mu2):
       e^{-T1} dT1 . dmu1/2 . e^{-s} ds . dmu2/2 1[mu2 >= mu_a] e^{-T2/mu2} . omega0^2,   T2 = T1 - mu1 s inside (0, tau),
       v~ = [(mu1 + 1) v(T1) + (mu2 - mu1) v(T2)] / 2        (Eq. 4 per event, launch direction mu0 = -1),
    v(T) the canonical depth table (T linear in v inside a bin, R24)."""
    tau = c.tau_ext
    nd = c.T_edge.size - 1
    v_edge = c.v_max - np.arange(nd + 1) * (c.v_max - c.v_fs) / nd
    v_of = lambda T: np.interp(T, c.T_edge, v_edge)
    x1, w1 = np.polynomial.legendre.leggauss(n1)
    T1 = 0.5 * tau * (x1 + 1.0); wT1 = 0.5 * tau * w1 * np.exp(-T1)
    xm, wm = np.polynomial.legendre.leggauss(nm)
    xs, ws = np.polynomial.legendre.leggauss(ns)
    xs, ws = 0.5 * (xs + 1.0), 0.5 * ws                                   # on [0, 1]
    x2, w2 = np.polynomial.legendre.leggauss(n2)
    mu2 = mu_a + 0.5 * (1.0 - mu_a) * (x2 + 1.0); wmu2 = 0.5 * (1.0 - mu_a) * w2 * 0.5
    vt_all, wt_all = [], []
    for sign in (+1.0, -1.0):                                            # second flight up (T2 < T1) / down (T2 > T1)
        mu1 = sign * 0.5 * (xm + 1.0); wmu1 = 0.5 * wm * 0.5             # |mu1| on (0, 1), density 1/2
        room = (T1 if sign > 0 else tau - T1)[:, None] / np.abs(mu1)[None, :]       # optical path to the boundary
        smax = np.minimum(room, 60.0)
        s = smax[:, :, None] * xs[None, None, :]
        wseg = smax[:, :, None] * ws[None, None, :] * np.exp(-s)
        T2 = T1[:, None, None] - mu1[None, :, None] * s
        base = wT1[:, None, None] * wmu1[None, :, None] * wseg * omega0 ** 2
        va = 0.5 * (mu1 + 1.0)[None, :, None] * v_of(T1)[:, None, None]
        v2 = v_of(T2)
        for m2, wq in zip(mu2, wmu2):
            vt_all.append((va + 0.5 * (m2 - mu1)[None, :, None] * v2).ravel())
            wt_all.append((base * wq * np.exp(-T2 / m2)).ravel())
    return np.concatenate(vt_all), np.concatenate(wt_all)


def test_double_scattering_spectrum_with_a_velocity_profile_P20(cfg2_oracle_cloud):
    """The part of the multiple-scattering spectrum that has a closed form although the particles move with a velocity
    PROFILE: histories of exactly two particle events (isotropic phase function, absorbing surface).  Transport (two free
    flights and the exit flight in a depth-dependent extinction), the per-event Doppler sum (Eq. 4) with the
    velocity taken at each event's own depth, implicit capture and the aperture all enter; the expectation is a 4-D
    Gauss-Legendre quadrature with no random number in it.  Compared: total weight, first three moments of v~, and a coarse
    histogram."""
    K = cfg2_oracle_cloud.phase.shape[1] - 1
    c = dataclasses.replace(cfg2_oracle_cloud, surface_reflectivity=0.0, phase=cloud.isotropic_quantile_table(K)[None, :])
    om = float(c.omega0[0])
    n = 4_000_000
    omega_sr = 2.0                                                        # a wide aperture: 4 % of the histories qualify
    mu_a = 1.0 - omega_sr / (2.0 * math.pi)
    r = mc.run(c, _run_opts(n, aperture_sr=omega_sr), trace=True)
    t = r.trace
    sel = (t["fate"] == 0) & (t["n_scatter"] == 2) & (t["n_reflect"] == 0)
    assert sel.sum() > 100_000
    assert np.allclose(t["w"][sel], om ** 2, rtol=1e-12)                  # implicit capture: two albedos
    vt, wt = _double_scatter_quadrature(c, om, mu_a)
    vt_b, wt_b = _double_scatter_quadrature(c, om, mu_a, n1=160, nm=80, ns=64, n2=8)    # the rule has converged
    for k in range(4):
        assert float(np.sum(wt_b * vt_b ** k)) == pytest.approx(float(np.sum(wt * vt ** k)), rel=2e-4)
    w_mc, v_mc = t["w"][sel], t["vt"][sel]
    W0 = float(wt.sum())
    # number of selected histories ~ Binomial(n, W0 / om^2)
    p_sel = W0 / om ** 2
    assert sel.sum() == pytest.approx(n * p_sel, abs=5 * math.sqrt(n * p_sel))
    for k in (1, 2, 3):                                                   # moments of v~ over the selected histories
        m_q = float(np.sum(wt * vt ** k)) / W0
        m_mc = float(np.mean(v_mc ** k))
        sig = float(np.std(v_mc ** k)) / math.sqrt(sel.sum())
        assert m_mc == pytest.approx(m_q, abs=5 * sig + 2e-4 * m_q), k
    edges = np.linspace(0.0, 6000.0, 25)                                  # 250 m/s bins: the rule's nodes are dense inside each
    h_q, _ = np.histogram(vt, bins=edges, weights=wt)
    h_mc, _ = np.histogram(v_mc, bins=edges, weights=w_mc)
    sig = np.sqrt(np.histogram(v_mc, bins=edges, weights=w_mc ** 2)[0])
    big = h_q * n > 2000 * om ** 2
    assert big.sum() >= 8
    assert np.all(np.abs(h_mc[big] - n * h_q[big]) <= 5 * sig[big] + 0.01 * n * h_q[big])
    # a Doppler sum that took both velocities at one depth, or dropped the second event, is far outside the band
    bad = float(np.sum(wt * 0.5 * (1.0 + np.full_like(vt, mu_a)) * 2000.0)) / W0
    assert abs(bad - float(np.mean(v_mc))) > 50 * float(np.std(v_mc)) / math.sqrt(sel.sum())
