"""ORACLE (test infrastructure, fp64) -- ejecta in a GAS environment: SURVEY.md 8(f) row f4.

Part of `oracle/`: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it; it never imports the CUDA
library and shares no code with it.

The paper treats the vacuum case only and names the gas case as future work in one sentence: "In a gas environment, the
particles slow down because of aerodynamic deceleration, and this introduces a series of changes to the PDV spectrum over time.
The particle deceleration is related to the particle size" (Conclusions).  It gives NO equation, so everything
below is a READING THAT IS NOT THE PAPER'S (R35-R38):

R35  The gas between the free surface and the shock it drives moves with the free surface (velocity v_fs, density rho_g).  A
     sphere of diameter d and density rho0 with velocity v feels the quasi-steady drag of a constant coefficient C_d on its
     velocity relative to the gas, u = v - v_fs:
         (pi/6) rho0 d^3 du/dt = -(1/2) C_d rho_g (pi/4) d^2 u^2     =>    du/dt = -u^2 / L,   L = 4 rho0 d / (3 C_d rho_g).
     Closed form for a particle ejected at t = 0 from the surface with relative velocity u0:
         u(t) = u0 / (1 + u0 t / L),      height above the free surface  zeta(t) = L ln(1 + u0 t / L).
     rho_g -> 0 (L -> infinity) is the paper's vacuum: u = u0, zeta = u0 t.  Small particles (small L) slow down first:
     "the particle deceleration is related to the particle size".
R36  Sizes are independent of the ejection velocity, so every size class c starts with the same mass
     distribution G in velocity (Eq. 20) and carries the optical thickness tau_ext P_c (Eq. 8, 10).  At time t the class-c
     particles above height zeta are those with u0 > u0_c(zeta) = (L_c/t)(e^{zeta/L_c} - 1), hence the vertical optical depth
     from the top
         T(zeta, t) = tau_ext sum_c P_c [1 - G(v_fs + u0_c(zeta))],
     the probability that an interaction at zeta hits class c,  P_c(zeta) = (dT_c/dzeta) / (dT/dzeta),  and the velocity of
     the class-c particle there,  v_c(zeta, t) = v_fs + (L_c/t)(1 - e^{-zeta/L_c}).  No particle is overtaken by the surface
     (u >= 0 always), so tau_ext does not change with time.
R37  Canonical discretisation (both sides use it, like R24): n_depth bins uniform in zeta on [0, zeta_top(t)], zeta_top =
     max_c L_c ln(1 + u_max t / L_c); T and every T_c exact at the edges, linear in zeta inside a bin (= piecewise-constant
     extinction AND piecewise-constant class probabilities per bin); the particle velocity is the continuous v_c at the
     interpolated zeta.  In the limit rho_g -> 0 this is exactly the vacuum discretisation R24 (uniform in v).
R38  The expected spectrum now DEPENDS on the snapshot time (reading R16 no longer holds): the tables belong to a
     (cloud, snapshot) unit, not to a cloud.
"""
from __future__ import annotations

import math

import numpy as np

from .cloud import OracleCloud, mass_cdf_exponential


def drag_length(diameter, density: float, gas_density: float, drag_coefficient: float):
    """L = 4 rho0 d / (3 C_d rho_g) per class; +inf in vacuum."""
    d = np.asarray(diameter, dtype=np.float64)
    if gas_density <= 0.0:
        return np.full(d.shape, np.inf)
    return 4.0 * density * d / (3.0 * drag_coefficient * gas_density)


def relative_velocity(u0, t: float, L):
    """u(t) = u0 / (1 + u0 t / L)."""
    return np.asarray(u0) / (1.0 + np.asarray(u0) * t / L)


def height(u0, t: float, L):
    """zeta(t) = L ln(1 + u0 t / L); u0 t in vacuum."""
    u0 = np.asarray(u0, dtype=np.float64)
    return np.where(np.isinf(L), u0 * t, L * np.log1p(u0 * t / np.where(np.isinf(L), 1.0, L)))


def initial_velocity_at(zeta, t: float, L):
    """u0 of the particle that is at height zeta at time t: (L/t)(e^{zeta/L} - 1)."""
    zeta = np.asarray(zeta, dtype=np.float64)
    return np.where(np.isinf(L), zeta / t, (np.where(np.isinf(L), 1.0, L) / t) * np.expm1(zeta / np.where(np.isinf(L), 1.0, L)))


def velocity_at_height(zeta, t: float, L):
    """Relative velocity of the class particle found at height zeta at time t: (L/t)(1 - e^{-zeta/L})."""
    zeta = np.asarray(zeta, dtype=np.float64)
    return np.where(np.isinf(L), zeta / t, -(np.where(np.isinf(L), 1.0, L) / t) * np.expm1(-zeta / np.where(np.isinf(L), 1.0, L)))


def build_tables(cloud: OracleCloud, params: dict, t: float, n_depth: int | None = None) -> dict:
    """Depth tables of one (cloud, snapshot) unit in a gas environment (readings R36, R37).

    params: the workload cloud dictionary (density, gas_density, drag_coefficient, profile, ...).
    Returns {"zeta_edge" [n+1] (zeta_top ... 0), "T_edge" [n+1] (0 ... tau_ext), "class_cum" [n][n_classes] cumulative class
    probabilities inside each bin (last column 1), "L" [n_classes], "t": t}.
    """
    n = int(n_depth or params.get("n_depth_bins", 1024))
    L = drag_length(cloud.diameters, params["density"], float(params.get("gas_density", 0.0)), float(params.get("drag_coefficient", 0.5)))
    v_fs, v_max = cloud.v_fs, cloud.v_max
    u_max = v_max - v_fs
    if cloud.profile_kind == 0:
        G = lambda v: np.clip(mass_cdf_exponential(np.minimum(v, v_max), v_fs, cloud.beta, v_max), 0.0, 1.0)
    else:
        pv = np.asarray(params["prof_v"], dtype=np.float64)
        pm = np.asarray(params["prof_cum_mass"], dtype=np.float64)
        G = lambda v: np.interp(np.minimum(v, v_max), pv, (pm - pm[0]) / (pm[-1] - pm[0]))
    zeta_top = float(np.max(height(u_max, t, L)))
    zeta = zeta_top * (1.0 - np.arange(n + 1) / n)
    zeta[-1] = 0.0
    # T_c at the edges: tau_ext P_c (1 - G(v_fs + u0_c(zeta)))
    Tc = np.empty((n + 1, cloud.n_classes))
    for c in range(cloud.n_classes):
        u0 = initial_velocity_at(zeta, t, L[c])
        Tc[:, c] = cloud.tau_ext * cloud.p_class[c] * (1.0 - G(v_fs + u0))
    Tc[-1, :] = cloud.tau_ext * cloud.p_class                       # zeta = 0: the whole class lies above
    T = Tc.sum(axis=1)
    T[0] = 0.0
    dTc = np.diff(Tc, axis=0)
    dT = dTc.sum(axis=1)
    with np.errstate(invalid="ignore", divide="ignore"):
        prob = np.where(dT[:, None] > 0.0, dTc / np.where(dT[:, None] > 0.0, dT[:, None], 1.0), cloud.p_class[None, :])
    cum = np.cumsum(prob, axis=1)
    cum[:, -1] = 1.0
    return {"zeta_edge": zeta, "T_edge": T, "class_cum": np.ascontiguousarray(cum), "L": L, "t": float(t)}
