"""Pins for the gas-environment variant of the oracle (oracle/gas.py readings R35-R38) -- CPU only.

The paper gives one sentence and no equation for this case, so the drag law is a reading that is NOT the paper's;
what is pinned here is that the oracle computes that reading correctly: the kinematics against a numerical integration of the
drag ODE, the tables against conservation laws and the vacuum limit, and the Monte-Carlo against closed-form / quadrature
single-backscatter spectra in which a wrong height, class probability or particle velocity shows up bin by bin.
"""
import dataclasses
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

import pdv_workloads as W
from oracle import cloud, gas, mc

from histcmp import compare, compare_to_expectation


def _run_opts(n, **kw):
    o = dict(W.config(1)["run"])
    o.update(n_photons=int(n), seed=777)
    o.update(kw)
    return o


# --------------------------------------------------------------------------------------------------------------- kinematics
@pytest.mark.parametrize("u0,L", [(4000.0, 0.05), (1500.0, 0.004), (300.0, 2.0)])
def test_drag_closed_form_solves_the_ode(u0, L):
    """du/dt = -u^2/L, dzeta/dt = u (R35), integrated numerically, against u0/(1 + u0 t/L) and L ln(1 + u0 t/L); and the two
    inverse maps used by the tables: u0 from (zeta, t), u from (zeta, t)."""
    t_end = 12e-6
    sol = solve_ivp(lambda t, y: [-y[0] ** 2 / L, y[0]], (0.0, t_end), [u0, 0.0], rtol=1e-12, atol=1e-15, dense_output=True)
    for t in (1e-7, 2e-6, 12e-6):
        u_num, z_num = sol.sol(t)
        assert float(gas.relative_velocity(u0, t, L)) == pytest.approx(u_num, rel=1e-9)
        z = float(gas.height(u0, t, L))
        assert z == pytest.approx(z_num, rel=1e-9)
        assert float(gas.initial_velocity_at(z, t, L)) == pytest.approx(u0, rel=1e-10)
        assert float(gas.velocity_at_height(z, t, L)) == pytest.approx(u_num, rel=1e-9)
    # vacuum: L = inf
    assert float(gas.height(u0, 3e-6, np.inf)) == u0 * 3e-6 and float(gas.velocity_at_height(0.012, 3e-6, np.inf)) == 0.012 / 3e-6
    # L = 4 rho0 d / (3 C_d rho_g): tin, 3 um, C_d 0.5, 5 kg/m^3
    assert float(gas.drag_length(3e-6, 7300.0, 5.0, 0.5)) == pytest.approx(4 * 7300 * 3e-6 / (3 * 0.5 * 5.0), rel=1e-15)
    assert np.isinf(gas.drag_length(3e-6, 7300.0, 0.0, 0.5))


# --------------------------------------------------------------------------------------------------------------- tables
@pytest.fixture(scope="module")
def cfg3_gas():
    params = dict(W.config(2)["clouds"][0], gas_density=5.0, drag_coefficient=0.5)
    return params, cloud.build_cloud(params)


def test_tables_conserve_optical_thickness_and_reduce_to_vacuum(cfg3_gas):
    params, c = cfg3_gas
    for t in (0.5e-6, 3e-6, 10e-6):
        g = gas.build_tables(c, params, t)
        T, z, cum = g["T_edge"], g["zeta_edge"], g["class_cum"]
        assert T[0] == 0.0 and T[-1] == pytest.approx(c.tau_ext, rel=1e-12)             # no particle is lost (R36)
        assert np.all(np.diff(T) >= 0.0) and np.all(np.diff(z) < 0.0) and z[-1] == 0.0
        assert np.all(np.diff(cum, axis=1) >= -1e-15) and np.all(cum[:, -1] == 1.0)
        # top of the cloud: the class that decelerates least, L ln(1 + u_max t / L)
        L = 4 * params["density"] * c.diameters / (3 * 0.5 * 5.0)
        assert z[0] == pytest.approx(np.max(L * np.log1p((c.v_max - c.v_fs) * t / L)), rel=1e-12)
        # per class: sum over bins of dT * P(class | bin) = tau_ext P_c
        prob = np.diff(np.concatenate([np.zeros((cum.shape[0], 1)), cum], axis=1), axis=1)
        assert np.allclose((np.diff(T)[:, None] * prob).sum(axis=0), c.tau_ext * c.p_class, rtol=1e-9)
        # size segregation: only the largest particles are found at the very top, the smallest sit lowest
        assert prob[0, -1] == pytest.approx(1.0) and prob[-1, 0] > prob[cum.shape[0] // 2, 0]
        if t >= 3e-6:
            assert prob[cum.shape[0] // 2, 0] == 0.0                 # no 0.7 um particle is left in the upper half of the cloud
    # rho_g -> 0: the vacuum tables of oracle/cloud.py (bins uniform in v, class probabilities P_c everywhere)
    thin = dict(params, gas_density=1e-9)
    g = gas.build_tables(c, thin, 3e-6)
    assert np.allclose(g["T_edge"], c.T_edge, rtol=1e-6, atol=1e-9 * c.tau_ext)
    assert np.allclose(g["class_cum"], np.cumsum(c.p_class)[None, :], atol=1e-6)
    v_edges = c.v_max - (c.v_max - c.v_fs) * np.arange(c.T_edge.size) / (c.T_edge.size - 1)
    assert np.allclose(c.v_fs + gas.velocity_at_height(g["zeta_edge"], 3e-6, g["L"][3]), v_edges, rtol=1e-6)


# --------------------------------------------------------------------------------------------------------------- Monte-Carlo
def _delta_back(c, p_class=None, omega0=None, diameters=None):
    """All classes scatter straight back (phase function = delta at theta = pi); black surface."""
    K = c.phase.shape[1] - 1
    n = len(diameters) if diameters is not None else c.n_classes
    kw = dict(phase=-np.ones((n, K + 1)), surface_reflectivity=0.0)
    if diameters is not None:
        kw.update(diameters=np.asarray(diameters), number_weights=np.full(n, 1.0 / n), k_ext=np.full(n, c.k_ext[0]),
                  k_sca=np.asarray(omega0) * c.k_ext[0], g=-np.ones(n), omega0=np.asarray(omega0, dtype=float),
                  p_class=np.asarray(p_class, dtype=float))
    return dataclasses.replace(c, **kw)


def test_single_backscatter_spectrum_of_one_size_in_gas_closed_form(cfg2_oracle_cloud):
    """One size class, all-backward scattering, single-scatter-only, R = 0, tiny aperture: every tallied photon carries the
    velocity v of its scatterer (pin P2), and with the drag law inverted in closed form,
        u = v - v_fs,   u0 = u / (1 - u t / L),   T(v) = tau_ext (1 - G(v_fs + u0)),
        H_k / N = omega0 / 2 [exp(-2 T(v_{k+1})) - exp(-2 T(v_k))].
    The spectrum is squeezed towards v_fs as t grows; its upper edge is v_fs + u_max / (1 + u_max t / L)."""
    params = dict(W.config(1)["clouds"][0], gas_density=8.0, drag_coefficient=0.5)
    c = _delta_back(cfg2_oracle_cloud)
    L = 4 * params["density"] * c.diameters[0] / (3 * 0.5 * 8.0)
    n = 1_500_000
    edges = np.linspace(0.0, 6000.0, 513)
    E = math.exp(-c.beta * (c.v_max / c.v_fs - 1.0))
    tops = []
    for t in (1e-6, 6e-6):
        g = gas.build_tables(c, params, t)
        r = mc.run(c, _run_opts(n, single_scatter_only=1, aperture_sr=1e-3), gas=g, trace=True)
        u_top = (c.v_max - c.v_fs) / (1.0 + (c.v_max - c.v_fs) * t / L)
        u = np.clip(edges - c.v_fs, 0.0, u_top)
        u0 = u / (1.0 - u * t / L)
        Tk = c.tau_ext * (np.exp(-c.beta * u0 / c.v_fs) - E) / (1.0 - E)
        Tk[edges >= c.v_fs + u_top] = 0.0
        expected = 0.5 * float(c.omega0[0]) * (np.exp(-2 * Tk[1:]) - np.exp(-2 * Tk[:-1]))
        res = compare_to_expectation(r.hist, r.hist2, n, expected)
        assert res["worst"] < 5.0 and res["ndf"] > 60, (t, res["worst"])
        det = r.trace[(r.trace["fate"] == 0) & (r.trace["w"] > 0)]
        assert det["vt"].max() <= c.v_fs + u_top + 1e-6 and det["vt"].min() >= c.v_fs - 1e-9
        tops.append(det["vt"].max())
    assert tops[1] < tops[0] - 200.0                    # the spectrogram's upper boundary comes down with time


def test_two_sizes_in_gas_against_quadrature(cfg2_oracle_cloud):
    """Two classes, 0.5 um (stopped quickly) and 20 um (almost ballistic), different hit probabilities and albedos, both
    scattering straight back:
        H_k / N = sum_c omega0_c int dzeta (-dT_c/dzeta) exp(-2 T(zeta)) 1[v_c(zeta) in bin k],
    T_c(zeta) = tau_ext P_c (1 - G(v_fs + (L_c/t)(e^{zeta/L_c} - 1))),  v_c = v_fs + (L_c/t)(1 - e^{-zeta/L_c})   (R36),
    by a midpoint rule in zeta.  A wrong per-bin class probability, class velocity or height puts the weight in other bins."""
    p_class, om, d = np.array([0.55, 0.45]), np.array([0.9, 0.5]), np.array([0.5e-6, 20e-6])
    c = _delta_back(cfg2_oracle_cloud, p_class, om, d)
    params = dict(W.config(1)["clouds"][0], gas_density=8.0, drag_coefficient=0.5)
    t = 4e-6
    g = gas.build_tables(c, params, t)
    n = 2_000_000
    r = mc.run(c, _run_opts(n, single_scatter_only=1, aperture_sr=1e-3), gas=g)
    L = 4 * params["density"] * d / (3 * 0.5 * 8.0)
    u_max = c.v_max - c.v_fs
    z_top = np.max(L * np.log1p(u_max * t / L))
    nz = 400_000
    z = (np.arange(nz) + 0.5) / nz * z_top
    E = math.exp(-c.beta * (c.v_max / c.v_fs - 1.0))

    def T_c(zz, k):
        u0 = (L[k] / t) * np.expm1(zz / L[k])
        G = np.clip((1.0 - np.exp(-c.beta * np.minimum(u0, u_max) / c.v_fs)) / (1.0 - E), 0.0, 1.0)
        return c.tau_ext * p_class[k] * (1.0 - G)

    dz = z_top / nz
    T = T_c(z, 0) + T_c(z, 1)
    expected = np.zeros(512)
    for k in range(2):
        dTc = T_c(z - 0.5 * dz, k) - T_c(z + 0.5 * dz, k)            # optical thickness of class k inside each slice
        v = c.v_fs + (L[k] / t) * (-np.expm1(-z / L[k]))
        h, _ = np.histogram(v, bins=512, range=(0.0, 6000.0), weights=om[k] * dTc * np.exp(-2.0 * T))
        expected += h
    res = compare_to_expectation(r.hist, r.hist2, n, expected, min_eff=50.0)
    assert res["worst"] < 5.0 and res["ndf"] > 40, res["worst"]
    assert r.stats["detected"] == pytest.approx(n * expected.sum(), abs=5 * math.sqrt(n * expected.sum()))
    # the small particles have piled up near v_fs: more than half of the detected weight lies below v_fs + 0.15 u_max
    k_cut = int((c.v_fs + 0.15 * u_max) / (6000.0 / 512))
    assert r.hist[:k_cut].sum() > 0.5 * r.hist.sum()


def test_spectrum_depends_on_time_in_gas_and_not_in_the_vacuum_limit(cfg3_gas):
    """Reading R38 against R16: with gas the spectra of two snapshot times differ far beyond the noise; with (almost) no gas the
    same two times are statistically indistinguishable, and equal to the vacuum run."""
    params, c = cfg3_gas
    n = 1_000_000
    a = mc.run(c, _run_opts(n, seed=1), gas=gas.build_tables(c, params, 1e-6))
    b = mc.run(c, _run_opts(n, seed=2), gas=gas.build_tables(c, params, 8e-6))
    res = compare(a.hist, a.hist2, n, b.hist, b.hist2, n)
    assert res["worst"] > 20.0 and res["chi2"] > 10 * res["ndf"]
    for r in (a, b):
        assert abs(r.conservation_residual()) < 1e-9 * n
    thin = dict(params, gas_density=1e-9)
    a0 = mc.run(c, _run_opts(n, seed=3), gas=gas.build_tables(c, thin, 1e-6))
    b0 = mc.run(c, _run_opts(n, seed=4), gas=gas.build_tables(c, thin, 8e-6))
    v = mc.run(c, _run_opts(n, seed=5))
    for x, y in ((a0, b0), (a0, v), (b0, v)):
        res = compare(x.hist, x.hist2, n, y.hist, y.hist2, n)
        assert res["worst"] < 5.0 and res["chi2"] < res["ndf"] + 5 * math.sqrt(2 * res["ndf"])
    # the optical structure does not change with time: same number of events per history (mean path), gas or not
    assert a.stats["particle_events"] / n == pytest.approx(v.stats["particle_events"] / n, rel=0.01)


def test_256_depth_bins_are_enough_for_the_gas_workload_at_1e8_histories():
    """The product runs 16 size classes in a gas with at most 256 depth bins (per-bin class thresholds: 16 x 1024 would not fit
    the shared memory of a block; include/pdv.h), where every vacuum workload uses 1024.  Two STORED oracle runs of the last
    snapshot of the row-f4 workload, 1e8 histories each, one with the workload's 256 bins and one with 1024
    (tests/golden/make_oracle_hists.py: f4gas_snap19, f4gas_snap19_nd1024; oracle against oracle, nothing of the CUDA path):
    their spectra agree bin by bin within 5 sigma of their own noise and their integrated rates to 5 sigma -- the
    discretisation error of 256 bins (reading R37) is below what 1e8 histories resolve."""
    from histcmp import load_golden, per_history_variance
    a, b = load_golden("f4gas_snap19"), load_golden("f4gas_snap19_nd1024")
    assert a.n_photons == b.n_photons == 10 ** 8 and a.run == b.run and a.tau_ext == pytest.approx(b.tau_ext, rel=1e-12)
    res = compare(a.hist, a.hist2, a.n_photons, b.hist, b.hist2, b.n_photons)
    assert res["ndf"] >= 200 and res["worst"] < 5.0, res["worst"]
    assert res["chi2"] < res["ndf"] + 6 * math.sqrt(2 * res["ndf"]) + 10, (res["chi2"], res["ndf"])
    for key in ("detected", "escaped", "absorbed_particles", "absorbed_surface"):
        x, y = a.stats[key] / a.n_photons, b.stats[key] / b.n_photons
        assert abs(x - y) < 5 * math.sqrt(max(x, 1e-12) / a.n_photons + max(y, 1e-12) / b.n_photons), (key, x, y)
    assert a.stats["particle_events"] / a.n_photons == pytest.approx(b.stats["particle_events"] / b.n_photons, rel=1e-3)
