"""ORACLE (test infrastructure, fp64) -- cloud optics and the canonical discretised tables.

Part of `oracle/`: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it; it
never imports the CUDA library and shares no code with it.

Follows SURVEY.md 8(c) steps 1-3 (readings listed in DESIGN.md):

* size classes (d_c, w_c), number weighted; `lognormal_classes` discretises Eq. 21
* mass-extinction coefficient kappa = 3 sum w d^2 K_ext / (2 rho0 sum w d^3), tau_ext = kappa m0
  (Eq. 10); class hit probability P_c = w_c d_c^2 K_ext,c / sum (Eq. 8)
* single-scattering albedo omega0_c = K_sca/K_ext (Eq. 11)
* canonical discretised phase function D_K: M[k] = F^-1(k/K), F the CDF of |S1|^2+|S2|^2 in
  mu = cos(theta) measured from mu = -1 (Eq. 13)
* mass CDF in velocity of Eq. 20 truncated to [v_fs, v_max] and renormalised,
  vertical optical depth from the top T(v) = tau_ext (1 - G(v)), tabulated at n_depth+1 velocity
  edges uniform in v and taken linear in v inside a bin (piecewise-constant extinction per bin).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
from scipy import integrate, special

from . import mie


def lognormal_classes(d_median: float, sigma_ln: float, n: int = 16):
    """Discretise the log-normal number distribution Eq. 21 into n classes.

    n bins of equal width in x = ln(d/d_m)/sigma over [-3, 3 + 3 sigma]; representative diameter at
    the bin centre in x; weight = standard-normal mass of the bin, renormalised to sum 1.
    """
    if sigma_ln == 0.0:
        return np.array([d_median]), np.array([1.0])
    edges = np.linspace(-3.0, 3.0 + 3.0 * sigma_ln, n + 1)
    centres = 0.5 * (edges[:-1] + edges[1:])
    cdf = special.ndtr(edges)
    w = np.diff(cdf)
    w = w / w.sum()
    return d_median * np.exp(sigma_ln * centres), w


def phase_quantile_table(x: float, m: complex, K: int, n_theta: int | None = None) -> np.ndarray:
    """M[0..K] with M[k] = F^-1(k/K) for the Mie phase function of size parameter x.

    F(mu) = int_{-1}^{mu} I dmu' / int_{-1}^{1} I dmu',  I = |S1|^2+|S2|^2.  Integrated in theta
    (dmu = sin th dth) from th = pi down to th on a uniform grid with composite Simpson; inside a
    grid cell the integrand is taken linear, so F is locally quadratic and is inverted in closed form.
    """
    a, b = mie.coefficients(x, m)
    if n_theta is None:
        n_theta = int(max(20000, 400 * x)) * 2          # even number of intervals, >= 127 nodes per lobe
    # psi = pi - theta runs 0..pi, so mu = -cos(psi) increases with psi
    psi = np.linspace(0.0, math.pi, n_theta + 1)
    mu = -np.cos(psi)
    gfun = np.empty_like(psi)
    chunk = 20000
    for s in range(0, psi.size, chunk):
        gfun[s:s + chunk] = mie.intensity(a, b, mu[s:s + chunk]) * np.sin(psi[s:s + chunk])
    F = integrate.cumulative_simpson(gfun, x=psi, initial=0.0)
    F = F / F[-1]
    M = np.empty(K + 1)
    M[0], M[K] = -1.0, 1.0
    targets = np.arange(1, K) / K
    idx = np.searchsorted(F, targets, side="right") - 1          # F[idx] <= target < F[idx+1]
    idx = np.clip(idx, 0, n_theta - 1)
    h = psi[1] - psi[0]
    g0, g1 = gfun[idx], gfun[idx + 1]
    # local model: F(psi_i + s) = F_i + c (g0 s + (g1-g0) s^2 / (2h)),  c fixed by F_{i+1}
    dF = F[idx + 1] - F[idx]
    c = dF / (0.5 * (g0 + g1) * h)
    r = (targets - F[idx]) / c                                  # = g0 s + (g1-g0) s^2/(2h)
    aq = (g1 - g0) / (2.0 * h)
    disc = np.sqrt(np.maximum(g0 * g0 + 4.0 * aq * r, 0.0))
    s = np.where(np.abs(aq) * h > 1e-14 * (np.abs(g0) + np.abs(g1)), 2.0 * r / (g0 + disc), r / np.maximum(g0, 1e-300))
    s = np.clip(s, 0.0, h)
    M[1:K] = -np.cos(psi[idx] + s)
    return M


def isotropic_quantile_table(K: int) -> np.ndarray:
    """D_K of the uniform ("isotropic") phase function, Fig. 6 Case 2."""
    return np.linspace(-1.0, 1.0, K + 1)


def mass_cdf_exponential(v, v_fs: float, beta: float, v_max: float):
    """G(v): cumulative mass fraction of Eq. 20 truncated to [v_fs, v_max] and renormalised."""
    E = math.exp(-beta * (v_max / v_fs - 1.0))
    return (1.0 - np.exp(-beta * (np.asarray(v) / v_fs - 1.0))) / (1.0 - E)


@dataclass
class OracleCloud:
    """Everything the oracle Monte-Carlo needs, all float64."""
    diameters: np.ndarray
    number_weights: np.ndarray
    k_ext: np.ndarray
    k_sca: np.ndarray
    g: np.ndarray
    omega0: np.ndarray            # per class K_sca/K_ext
    p_class: np.ndarray           # class hit probabilities
    kappa: float                  # m^2/kg
    tau_ext: float
    v_fs: float
    v_max: float
    beta: float
    profile_kind: int
    phase: np.ndarray             # [n_classes, K+1]
    T_edge: np.ndarray            # [n_depth+1]; T_edge[j] at v = v_max - j dv; T_edge[0]=0, T_edge[-1]=tau_ext
    surface_reflectivity: float
    surface_model: int
    sauter_diameter: float
    extra: dict = field(default_factory=dict)

    @property
    def n_classes(self):
        return len(self.diameters)


def build_cloud(params: dict, *, phase_override: np.ndarray | None = None) -> OracleCloud:
    """Build an OracleCloud from a workload cloud dictionary (see pdv_workloads._cloud)."""
    if "lognormal" in params:
        ln = params["lognormal"]
        d, w = lognormal_classes(ln["d_median"], ln["sigma_ln"], ln["n_classes"])
    else:
        d = np.asarray(params["diameters"], dtype=np.float64)
        w = np.asarray(params["number_weights"], dtype=np.float64)
        w = w / w.sum()
    m = complex(params["m_re"], params["m_im"])
    lam = params["wavelength"]
    K = int(params.get("n_phase_bins", 1024))
    n_depth = int(params.get("n_depth_bins", 1024))
    eff = np.array([mie.efficiencies(math.pi * di / lam, m) for di in d])
    k_ext, k_sca, g = eff[:, 0], eff[:, 1], eff[:, 3]
    sum_ext = np.sum(w * d**2 * k_ext)
    kappa = 3.0 * sum_ext / (2.0 * params["density"] * np.sum(w * d**3))
    tau_ext = kappa * params["area_mass"]
    p_class = w * d**2 * k_ext / sum_ext
    if phase_override is not None:
        phase = np.asarray(phase_override, dtype=np.float64).reshape(len(d), -1)
    else:
        cache = {}
        rows = []
        for di in d:
            key = float(di)
            if key not in cache:
                cache[key] = phase_quantile_table(math.pi * di / lam, m, K)
            rows.append(cache[key])
        phase = np.stack(rows)
    v_fs = params["v_fs"]
    v_max = params["vmax_ratio"] * v_fs
    v_edges = v_max - (v_max - v_fs) * np.arange(n_depth + 1) / n_depth
    kind = int(params.get("profile_kind", 0))
    if kind == 0:
        G = mass_cdf_exponential(v_edges, v_fs, params["beta"], v_max)
    else:
        pv = np.asarray(params["prof_v"], dtype=np.float64)
        pm = np.asarray(params["prof_cum_mass"], dtype=np.float64)
        G = np.interp(v_edges, pv, (pm - pm[0]) / (pm[-1] - pm[0]))
    T_edge = tau_ext * (1.0 - G)
    T_edge[0] = 0.0
    T_edge[-1] = tau_ext
    return OracleCloud(
        diameters=d, number_weights=w, k_ext=k_ext, k_sca=k_sca, g=g, omega0=k_sca / k_ext,
        p_class=p_class, kappa=float(kappa), tau_ext=float(tau_ext), v_fs=v_fs, v_max=v_max,
        beta=float(params.get("beta", 0.0)), profile_kind=kind, phase=phase, T_edge=T_edge,
        surface_reflectivity=float(params["surface_reflectivity"]), surface_model=int(params.get("surface_model", 0)),
        sauter_diameter=float(np.sum(w * d**3) / np.sum(w * d**2)),
    )
