"""Seeded synthetic workload definitions shared by the oracle tests, the CUDA tests and bench.py.

This module holds NONE of the method's arithmetic: it only names the physical inputs of the
BASELINE.json configs as plain numbers, in SI units.  Everything
derived from them (Mie efficiencies, size classes, tables, histograms) is computed independently
by `oracle/` (test infrastructure, fp64) and by the CUDA library (product path).  Neither of those
imports the other; both may be handed the dictionaries below by a test or by bench.py.

The paper's workloads are parametric tin-ejecta clouds (section II.C; Fig. 4
caption PAPER.md:215), so "synthetic" here means exactly what the paper simulates: no dataset is
involved.
"""
from __future__ import annotations

import copy

# Material / probe constants fixed by BASELINE.json (the paper gives neither the index of Sn at
# 1550 nm nor its density).
M_RE, M_IM = 2.5, 9.5            # complex refractive index m = 2.5 + 9.5i (Im > 0 absorbs)
WAVELENGTH = 1550e-9             # m   ("1550 mm" there is a typo)
DENSITY = 7300.0                 # kg/m^3
SURFACE_REFLECTIVITY = 0.6
APERTURE_SR = 0.1
N_PHASE_BINS = 1024
N_DEPTH_BINS = 1024

MG_CM2 = 1.0e-2                  # 1 mg/cm^2 in kg/m^2


def _cloud(area_mass_mg_cm2, beta, v_fs, *, diameter_um=None, lognormal=None, vmax_ratio=3.0):
    """One cloud description.  Exactly one of `diameter_um` (monodisperse) or
    `lognormal=(median_um, sigma_ln, n_classes)` is given."""
    c = dict(
        area_mass=area_mass_mg_cm2 * MG_CM2, density=DENSITY, v_fs=float(v_fs), beta=float(beta),
        vmax_ratio=float(vmax_ratio), m_re=M_RE, m_im=M_IM, wavelength=WAVELENGTH,
        surface_reflectivity=SURFACE_REFLECTIVITY, surface_model=0,
        n_phase_bins=N_PHASE_BINS, n_depth_bins=N_DEPTH_BINS,
    )
    if (diameter_um is None) == (lognormal is None):
        raise ValueError("give exactly one of diameter_um / lognormal")
    if diameter_um is not None:
        c["diameters"] = [diameter_um * 1e-6]
        c["number_weights"] = [1.0]
    else:
        med, sig, n = lognormal
        c["lognormal"] = dict(d_median=med * 1e-6, sigma_ln=float(sig), n_classes=int(n))
    return c


def _run(n_photons, seed, n_bins, v_hi, *, max_events=0, roulette_survival=0.1):
    return dict(n_photons=int(n_photons), seed=int(seed), n_bins=int(n_bins), v_lo=0.0, v_hi=float(v_hi),
                aperture_sr=APERTURE_SR, mode=0, max_events=int(max_events),
                roulette_survival=float(roulette_survival), single_scatter_only=0)


def config(index: int) -> dict:
    """BASELINE.json `configs[index]` as concrete inputs (index 0..4 = SURVEY config 1..5).

    Returns {"name", "clouds": [cloud...], "t_snap": [seconds...], "run": {...}}.
    """
    if index == 0:    # single-scatter dominated, 1e5 photons
        return dict(name="cfg1_thin_mono", clouds=[_cloud(0.1, 4.0, 2000.0, diameter_um=5.0)],
                    t_snap=[2.0e-6], run=_run(1e5, 1, 512, 6000.0))
    if index == 1:    # headline: multiple scattering, 1e8 photons
        return dict(name="cfg2_multi_mono", clouds=[_cloud(2.0, 4.0, 2000.0, diameter_um=5.0)],
                    t_snap=[3.0e-6], run=_run(1e8, 2, 512, 6000.0))
    if index == 2:    # polydisperse, 200 snapshots
        ts = [0.5e-6 + i * (10.0e-6 - 0.5e-6) / 199 for i in range(200)]
        return dict(name="cfg3_poly_spectrogram", clouds=[_cloud(5.0, 4.0, 2000.0, lognormal=(3.0, 0.5, 16))],
                    t_snap=ts, run=_run(1e8, 3, 512, 6000.0))
    if index == 3:    # 48-cloud sweep
        clouds = [_cloud(m0, beta, 2000.0, diameter_um=d)
                  for m0 in (0.5, 1, 2, 5, 10, 20) for d in (1, 2, 5, 10) for beta in (2, 6)]
        return dict(name="cfg4_sweep48", clouds=clouds, t_snap=[2.0e-6], run=_run(1e7, 4, 1024, 6000.0))
    if index == 4:    # optically thick stress case (velocity range 0..3 v_fs)
        return dict(name="cfg5_thick_poly", clouds=[_cloud(30.0, 4.0, 3000.0, lognormal=(1.0, 0.7, 16))],
                    t_snap=[2.0e-6], run=_run(1e9, 5, 2048, 9000.0, max_events=200, roulette_survival=0.1))
    raise IndexError(index)


def scaled(cfg: dict, n_photons: int, n_snap: int | None = None, n_clouds: int | None = None) -> dict:
    """Copy of `cfg` with fewer photons / snapshots / clouds (parity-test and CPU-baseline sizes)."""
    c = copy.deepcopy(cfg)
    c["run"]["n_photons"] = int(n_photons)
    if n_snap is not None:
        c["t_snap"] = c["t_snap"][:n_snap]
    if n_clouds is not None:
        c["clouds"] = c["clouds"][:n_clouds]
    return c


# The paper's own base case (Fig. 4 caption; sensitivity studies PAPER.md:233):
# beta=10, m0=20 mg/cm^2, d_m=1.5 um, sigma=0.5.  v_fs is not printed for the simulations; the
# experimental value 2013 m/s is of the same order as BASELINE.json's 2000 m/s.
def paper_base_case(n_photons=1e7, seed=7) -> dict:
    return dict(name="paper_fig4", clouds=[_cloud(20.0, 10.0, 2000.0, lognormal=(1.5, 0.5, 16))],
                t_snap=[2.0e-6], run=_run(n_photons, seed, 512, 6000.0))


# The paper's parameter studies around that base case (section III.A; Figs. 7-10) and the two
# optical thicknesses of Figs. 13-15 (tau0 = 23.4 <-> m0 = 20 mg/cm^2, d_m = 1.5 um; tau0 = 8.6 <->
# m0 = 10 mg/cm^2, d_m = 2.0 um; sigma = 0.5) over "a large range of velocity profiles".  The swept values are not
# printed in the text (they are in the figures); the ones below bracket the base case.  One launch runs a whole sweep.
PAPER_SWEEPS = {
    "fig7_beta": [dict(m0=20.0, beta=b, d_m=1.5, sigma=0.5) for b in (6.0, 8.0, 10.0, 12.0, 14.0)],
    "fig8_m0": [dict(m0=m, beta=10.0, d_m=1.5, sigma=0.5) for m in (2.0, 5.0, 10.0, 20.0, 40.0)],
    "fig9_dm": [dict(m0=20.0, beta=10.0, d_m=d, sigma=0.5) for d in (0.5, 1.0, 1.5, 2.0, 3.0)],
    "fig10_sigma": [dict(m0=20.0, beta=10.0, d_m=1.5, sigma=s) for s in (0.3, 0.4, 0.5, 0.6, 0.7)],
    "fig13_15": [dict(m0=m, beta=b, d_m=d, sigma=0.5) for (m, d) in ((20.0, 1.5), (10.0, 2.0))
                 for b in (4.0, 6.0, 8.0, 10.0, 12.0, 16.0, 20.0)],
}


def paper_sweep(name: str, n_photons=1e7, seed=11, n_bins=1024, v_fs=2000.0) -> dict:
    """One of PAPER_SWEEPS as a multi-cloud workload; `points` keeps the swept parameters of each cloud."""
    pts = PAPER_SWEEPS[name]
    return dict(name=f"paper_{name}", points=copy.deepcopy(pts),
                clouds=[_cloud(p["m0"], p["beta"], v_fs, lognormal=(p["d_m"], p["sigma"], 16)) for p in pts],
                t_snap=[2.0e-6], run=_run(n_photons, seed, n_bins, 3.0 * v_fs))


# SURVEY.md 8(f) row f4 (the paper's stated future work; readings R35-R38 are NOT the paper's): config 3's
# 16-class cloud in a gas that moves with the free surface.  The depth tables depend on the snapshot time, so every snapshot is
# a unit with its own device image; 20 snapshots x 1e7 photons.  Gas density 5 kg/m^3, drag coefficient 0.5, 256 depth bins
# (the values of tests/test_gpu_gas.py).
def gas_spectrogram(n_photons=1e7, n_snap=20, seed=13) -> dict:
    ts = [0.5e-6 + i * (10.0e-6 - 0.5e-6) / max(n_snap - 1, 1) for i in range(n_snap)]
    cl = dict(_cloud(5.0, 4.0, 2000.0, lognormal=(3.0, 0.5, 16)), gas_density=5.0, drag_coefficient=0.5, n_depth_bins=256)
    return dict(name="f4_gas_spectrogram", clouds=[cl], t_snap=ts, run=_run(n_photons, seed, 512, 6000.0))

