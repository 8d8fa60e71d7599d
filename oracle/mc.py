"""ORACLE (test infrastructure, fp64) -- Python driver of the plain C Monte-Carlo `pdv_oracle_mc.c`.

Part of `oracle/`: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it; it
never imports the CUDA library.  `build()` compiles the C file with gcc (-O2, no fast-math) into
oracle/_build/libpdv_oracle.so; `run()` marshals an `OracleCloud` and run options into the C struct.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass

import numpy as np

from . import mie
from .cloud import OracleCloud

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pdv_oracle_mc.c")
_BUILD = os.path.join(_HERE, "_build")
_SO = os.path.join(_BUILD, "libpdv_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle C code (gcc -O2 -std=c11, no fast-math).  Returns the .so path."""
    os.makedirs(_BUILD, exist_ok=True)
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-D_GNU_SOURCE", "-fPIC", "-shared", "-pthread",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


class _Params(C.Structure):
    _fields_ = [
        ("n_classes", C.c_int32), ("K", C.c_int32), ("n_depth", C.c_int32),
        ("phase", C.POINTER(C.c_double)), ("p_cum", C.POINTER(C.c_double)),
        ("omega0", C.POINTER(C.c_double)), ("T_edge", C.POINTER(C.c_double)),
        ("v_fs", C.c_double), ("v_max", C.c_double), ("tau_ext", C.c_double),
        ("analytic_profile", C.c_int32), ("beta", C.c_double),
        ("R", C.c_double), ("surface_model", C.c_int32),
        ("exact_mie", C.c_int32), ("mie_nmax", C.POINTER(C.c_int32)), ("mie_ab", C.POINTER(C.c_double)),
        ("mie_stride", C.c_int32), ("mie_gmax", C.POINTER(C.c_double)),
        ("n_bins", C.c_int32), ("v_lo", C.c_double), ("v_hi", C.c_double), ("mu_aperture", C.c_double),
        ("mode", C.c_int32), ("max_events", C.c_int32), ("p_roulette", C.c_double),
        ("single_scatter_only", C.c_int32), ("rng_mode", C.c_int32), ("seed", C.c_uint64),
        ("stream", C.c_uint32), ("launch_model", C.c_int32),
        ("gas", C.c_int32), ("zeta_edge", C.POINTER(C.c_double)), ("class_cum", C.POINTER(C.c_double)),
        ("gas_L", C.POINTER(C.c_double)), ("t_snap", C.c_double),
    ]


class _Stats(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("detected", "underflow", "overflow", "escaped", "absorbed_particles",
                                          "absorbed_surface", "roulette_killed", "roulette_gained", "truncated")] + \
               [(n, C.c_uint64) for n in ("histories", "particle_events", "surface_reflections",
                                          "max_events_in_history")]


TRACE_DTYPE = np.dtype([("vt", "f8"), ("vt_leg", "f8"), ("w", "f8"), ("mu_exit", "f8"),
                        ("fate", "i4"), ("n_scatter", "i4"), ("n_reflect", "i4")], align=True)


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_mc_run.restype = C.c_int
        _lib.oracle_mc_run.argtypes = [C.POINTER(_Params), C.c_uint64, C.c_uint64, C.c_int,
                                       C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(_Stats), C.c_void_p]
        _lib.oracle_philox4x32_10.restype = None
        _lib.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        _lib.oracle_rotate.restype = None
        _lib.oracle_rotate.argtypes = [C.POINTER(C.c_double), C.c_double, C.c_double]
    return _lib


def philox4x32_10(counter, key):
    """The oracle's Philox4x32-10 block function (4 counter words, 2 key words) -> 4 output words."""
    lib = _load()
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in counter])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib.oracle_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def rotate(u, cos_theta: float, phi: float):
    """Eq. 16/17 rotation of the direction cosines u by (theta, phi) -- exposed for pin P6."""
    lib = _load()
    a = (C.c_double * 3)(*u)
    lib.oracle_rotate(a, cos_theta, phi)
    return np.array(a[:])


def aperture_mu(aperture_sr: float) -> float:
    """On-axis cone of solid angle Omega: mu >= 1 - Omega/(2 pi)  (reading R6)."""
    return 1.0 - aperture_sr / (2.0 * math.pi)


@dataclass
class OracleResult:
    hist: np.ndarray
    hist2: np.ndarray
    stats: dict
    trace: np.ndarray | None
    n_photons: int

    def conservation_residual(self) -> float:
        s = self.stats
        return (s["detected"] + s["underflow"] + s["overflow"] + s["escaped"] + s["absorbed_particles"]
                + s["absorbed_surface"] + s["roulette_killed"] - s["roulette_gained"] + s["truncated"]
                - self.n_photons)


def run(cloud: OracleCloud, run_opts: dict, *, n_photons: int | None = None, first_id: int = 0, stream: int = 0,
        seed: int | None = None, rng_mode: int = 0, n_threads: int | None = None, analytic_profile: bool = False,
        exact_mie: dict | None = None, trace: bool = False, launch_model: int = 0, gas: dict | None = None) -> OracleResult:
    """Run the oracle Monte-Carlo for one (cloud, snapshot) unit.

    run_opts: the "run" dictionary of a pdv_workloads config (n_bins, v_lo, v_hi, aperture_sr, mode,
    max_events, roulette_survival, single_scatter_only, n_photons, seed).
    exact_mie: {"m": complex, "wavelength": float} switches theta sampling to acceptance-rejection
    on the exact Mie function; requires rng_mode 0.
    launch_model 1: diffuse (Lambertian) illumination of the cloud top instead of the paper's collimated beam -- exists
    only for the invariance pin of the multiple-scattering core (tests/test_oracle_mc.py), rng_mode 0.
    gas: the tables of oracle/gas.py::build_tables for this (cloud, snapshot) unit -- ejecta decelerated by a gas
    (SURVEY.md 8(f) row f4); None: the paper's vacuum.
    """
    lib = _load()
    n = int(run_opts["n_photons"] if n_photons is None else n_photons)
    if n_threads is None:
        n_threads = os.cpu_count() or 1
    phase = np.ascontiguousarray(cloud.phase, dtype=np.float64)
    p_cum = np.ascontiguousarray(np.cumsum(cloud.p_class), dtype=np.float64)
    p_cum[-1] = 1.0
    omega0 = np.ascontiguousarray(cloud.omega0, dtype=np.float64)
    T_edge = np.ascontiguousarray(cloud.T_edge if gas is None else gas["T_edge"], dtype=np.float64)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    p = _Params()
    p.n_classes, p.K, p.n_depth = cloud.n_classes, phase.shape[1] - 1, T_edge.size - 1
    p.phase, p.p_cum, p.omega0, p.T_edge = dp(phase), dp(p_cum), dp(omega0), dp(T_edge)
    p.v_fs, p.v_max, p.tau_ext = cloud.v_fs, cloud.v_max, cloud.tau_ext
    p.analytic_profile, p.beta = int(analytic_profile), cloud.beta
    p.R, p.surface_model = cloud.surface_reflectivity, cloud.surface_model
    keep = []
    if exact_mie is not None:
        if rng_mode != 0:
            raise ValueError("exact-Mie rejection needs rng_mode 0")
        m, lam = exact_mie["m"], exact_mie["wavelength"]
        coefs = [mie.coefficients(math.pi * d / lam, m) for d in cloud.diameters]
        stride = max(len(a) for a, _ in coefs)
        ab = np.zeros((cloud.n_classes, 4, stride))
        nmax = np.zeros(cloud.n_classes, dtype=np.int32)
        gmax = np.zeros(cloud.n_classes)
        for c, (a, b) in enumerate(coefs):
            nmax[c] = len(a)
            ab[c, 0, :len(a)], ab[c, 1, :len(a)], ab[c, 2, :len(a)], ab[c, 3, :len(a)] = a.real, a.imag, b.real, b.imag
            th = np.linspace(0.0, math.pi, 200001)
            gmax[c] = 1.02 * np.max(mie.intensity(a, b, np.cos(th)) * np.sin(th))
        keep += [ab, nmax, gmax]
        p.exact_mie, p.mie_stride = 1, stride
        p.mie_nmax = nmax.ctypes.data_as(C.POINTER(C.c_int32))
        p.mie_ab, p.mie_gmax = dp(ab), dp(gmax)
    p.n_bins, p.v_lo, p.v_hi = int(run_opts["n_bins"]), float(run_opts["v_lo"]), float(run_opts["v_hi"])
    p.mu_aperture = aperture_mu(run_opts["aperture_sr"])
    p.mode, p.max_events = int(run_opts.get("mode", 0)), int(run_opts.get("max_events", 0))
    p.p_roulette = float(run_opts.get("roulette_survival", 0.1))
    p.single_scatter_only = int(run_opts.get("single_scatter_only", 0))
    p.rng_mode, p.seed, p.stream = int(rng_mode), int(run_opts["seed"] if seed is None else seed), int(stream)
    if launch_model and rng_mode != 0:
        raise ValueError("launch_model 1 (diffuse illumination, pins only) needs rng_mode 0")
    p.launch_model = int(launch_model)
    if gas is not None:
        if analytic_profile:
            raise ValueError("the closed-form depth profile exists for the vacuum case only")
        g_zeta = np.ascontiguousarray(gas["zeta_edge"], dtype=np.float64)
        g_cum = np.ascontiguousarray(gas["class_cum"], dtype=np.float64)
        g_L = np.ascontiguousarray(gas["L"], dtype=np.float64)
        if g_zeta.size != T_edge.size or g_cum.shape != (T_edge.size - 1, cloud.n_classes) or g_L.size != cloud.n_classes:
            raise ValueError("gas tables do not match the cloud")
        keep += [g_zeta, g_cum, g_L]
        p.gas, p.zeta_edge, p.class_cum, p.gas_L, p.t_snap = 1, dp(g_zeta), dp(g_cum), dp(g_L), float(gas["t"])
    hist = np.zeros(p.n_bins)
    hist2 = np.zeros(p.n_bins)
    st = _Stats()
    tr = np.zeros(n, dtype=TRACE_DTYPE) if trace else None
    rc = lib.oracle_mc_run(C.byref(p), int(first_id), n, int(n_threads), dp(hist), dp(hist2), C.byref(st),
                           tr.ctypes.data if trace else None)
    if rc != 0:
        raise MemoryError("oracle_mc_run failed")
    stats = {name: getattr(st, name) for name, _ in _Stats._fields_}
    return OracleResult(hist, hist2, stats, tr, n)
