"""ctypes binding of libpdv_b200.so (include/pdv.h).  Argument marshalling only: every step of the hot path
runs in the CUDA kernels behind the C-ABI.  There is no CPU fallback; if the shared library is missing
the import fails loudly (build it with `python -m paper_2012_00963_b200.build`).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpdv_b200.so")

PDV_OK, PDV_E_INVALID, PDV_E_NOMEM, PDV_E_CUDA, PDV_E_UNSUPPORTED = range(5)
PDV_MAX_CLASSES = 32
PDV_MAX_BINS = 8192
PDV_STATIC_SCRATCH_BYTES = 2 << 20

EXPORTS = ("pdv_lognormal_classes", "pdv_cloud_create", "pdv_cloud_destroy", "pdv_cloud_get_info",
           "pdv_estimated_flights", "pdv_cloud_get_tables", "pdv_cloud_get_image", "pdv_cloud_gas_tables", "pdv_mc_run", "pdv_mc_run_static", "pdv_mc_trace", "pdv_spectrogram", "pdv_spectrum_peaks", "pdv_phase_sampling_check", "pdv_philox_blocks", "pdv_issue_peaks",
           "pdv_last_launch_info", "pdv_launch_info_on_stream", "pdv_last_error", "pdv_version")


class PdvError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"pdv status {status}: {message}")
        self.status = status


class CloudParams(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("area_mass", C.c_double), ("density", C.c_double), ("v_fs", C.c_double),
                ("profile_kind", C.c_int32), ("beta", C.c_double), ("vmax_ratio", C.c_double),
                ("n_prof", C.c_int32), ("prof_v", C.POINTER(C.c_double)), ("prof_cum_mass", C.POINTER(C.c_double)),
                ("n_classes", C.c_int32), ("diameter", C.POINTER(C.c_double)), ("number_weight", C.POINTER(C.c_double)),
                ("m_re", C.c_double), ("m_im", C.c_double), ("wavelength", C.c_double),
                ("surface_reflectivity", C.c_double), ("surface_model", C.c_int32),
                ("n_phase_bins", C.c_int32), ("n_depth_bins", C.c_int32), ("phase_model", C.c_int32),
                ("depth_model", C.c_int32), ("gas_density", C.c_double), ("drag_coefficient", C.c_double)]


class CloudInfo(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("n_classes", C.c_int32), ("n_phase_bins", C.c_int32),
                ("n_depth_bins", C.c_int32), ("on_device", C.c_int32), ("tau_ext", C.c_double), ("kappa", C.c_double),
                ("sauter_diameter", C.c_double), ("v_fs", C.c_double), ("v_max", C.c_double),
                ("mean_albedo", C.c_double), ("mean_g", C.c_double)]


class RunOpts(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("n_bins", C.c_int32), ("v_lo", C.c_double), ("v_hi", C.c_double),
                ("aperture_sr", C.c_double), ("mode", C.c_int32), ("max_events", C.c_int32),
                ("roulette_survival", C.c_double), ("single_scatter_only", C.c_int32),
                ("first_photon_id", C.c_uint64), ("output_on_device", C.c_int32), ("blocks_per_sm", C.c_int32),
                ("threads_per_block", C.c_int32), ("launch_model", C.c_int32),
                ("unit_streams", C.POINTER(C.c_uint32))]


STAT_FLOATS = ("detected", "underflow", "overflow", "escaped", "absorbed_particles", "absorbed_surface",
               "roulette_killed", "roulette_gained", "truncated")
STAT_INTS = ("histories", "particle_events", "surface_reflections", "max_events_in_history")
STATS_DTYPE = np.dtype([(n, "f8") for n in STAT_FLOATS] + [(n, "u8") for n in STAT_INTS])
TRACE_DTYPE = np.dtype([("vt", "f4"), ("weight", "f4"), ("mu_exit", "f4"), ("fate", "i4"), ("n_scatter", "i4"),
                        ("n_reflect", "i4")])
PEAK_DTYPE = np.dtype([("x_peak", "f8"), ("i_peak", "f8"), ("curvature", "f8"), ("k_peak", "i4"), ("status", "i4"),
                       ("beta_eq35", "f8"), ("tau0_eq35", "f8")])


class ImageLayout(C.Structure):
    _fields_ = [("struct_size", C.c_size_t)] + [(n, C.c_uint32) for n in (
        "image_bytes", "n_classes", "n_phase_bins", "log2_phase_bins", "n_depth_bins", "off_phase", "off_rows", "off_thr", "off_thr24",
        "off_albedo", "off_guide", "n_guide", "guide_base", "guide_shift", "depth_bisect", "off_cguide", "cguide_cells", "cguide_shift",
        "cguide_flagged", "frac_mask")] + [(n, C.c_float) for n in ("tau_ext_ln2", "half_v_fs", "surface_reflectivity")]


class PhaseCheck(C.Structure):
    _fields_ = [("sum_cos_table", C.c_double), ("sum_cos_exact", C.c_double), ("i_max", C.c_double),
                ("n_trials", C.c_uint64), ("n_bound_violations", C.c_uint64)]


class PeakOpts(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("smooth_half", C.c_int32), ("smooth_passes", C.c_int32),
                ("fit_half", C.c_int32), ("pad", C.c_int32), ("x_min", C.c_double), ("x_max", C.c_double)]


_lib = None


def lib() -> C.CDLL:
    """Loads the shared library (once).  Raises if it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2012_00963_b200.build` "
                              "(the CUDA library is the only implementation; there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        dp, vp = C.POINTER(C.c_double), C.c_void_p
        L.pdv_lognormal_classes.argtypes = [C.c_double, C.c_double, C.c_int32, dp, dp, C.POINTER(C.c_int32)]
        L.pdv_cloud_create.argtypes = [C.POINTER(CloudParams), C.POINTER(vp)]
        L.pdv_cloud_destroy.argtypes = [vp]
        L.pdv_cloud_destroy.restype = None
        L.pdv_cloud_get_info.argtypes = [vp, C.POINTER(CloudInfo)]
        L.pdv_estimated_flights.argtypes = [vp, C.POINTER(RunOpts), dp]
        L.pdv_cloud_get_tables.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.pdv_cloud_get_image.argtypes = [vp, C.POINTER(ImageLayout), vp, C.c_size_t]
        L.pdv_cloud_gas_tables.argtypes = [vp, C.c_double, vp, vp, vp, vp]
        L.pdv_mc_run.argtypes = [C.POINTER(vp), C.c_int32, dp, C.c_int32, C.c_uint64, C.c_uint64, C.POINTER(RunOpts),
                                 vp, vp, vp, vp]
        L.pdv_mc_run_static.argtypes = L.pdv_mc_run.argtypes
        L.pdv_mc_trace.argtypes = [vp, C.c_uint32, C.c_uint64, C.c_uint64, C.POINTER(RunOpts), vp, vp, vp, vp, vp]
        L.pdv_spectrogram.argtypes = [vp, C.c_int32, C.c_int32, C.c_uint64, C.c_double, C.c_double, C.c_int32,
                                      C.c_float, vp, C.c_int32, vp]
        L.pdv_spectrum_peaks.argtypes = [vp, C.c_int32, C.c_int32, C.c_uint64, C.c_double, C.c_double, vp,
                                         C.POINTER(PeakOpts), vp, C.c_int32, vp]
        L.pdv_phase_sampling_check.argtypes = [vp, C.c_int32, C.c_uint64, C.c_uint64, C.c_int32, vp, vp, C.POINTER(PhaseCheck), vp]
        L.pdv_philox_blocks.argtypes = [vp, C.c_int32, C.c_uint64, vp, vp, vp]
        L.pdv_issue_peaks.argtypes = [C.c_double, dp, dp, dp, C.POINTER(C.c_int32), vp]
        L.pdv_last_launch_info.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_float), C.POINTER(C.c_int32),
                                           C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.pdv_launch_info_on_stream.argtypes = [vp] + L.pdv_last_launch_info.argtypes
        L.pdv_last_error.restype = C.c_char_p
        L.pdv_version.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("pdv_cloud_destroy", "pdv_last_error", "pdv_version"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(status: int):
    if status != PDV_OK:
        raise PdvError(status, lib().pdv_last_error().decode())


def pdv_version() -> str:
    return lib().pdv_version().decode()


def pdv_lognormal_classes(d_median: float, sigma_ln: float, n: int = 16):
    """-> (diameters[n], number_weights[n]) of Eq. 21 discretised (see include/pdv.h)."""
    d = np.zeros(max(n, 1))
    w = np.zeros(max(n, 1))
    n_out = C.c_int32(0)
    dp = C.POINTER(C.c_double)
    _check(lib().pdv_lognormal_classes(d_median, sigma_ln, n, d.ctypes.data_as(dp), w.ctypes.data_as(dp), C.byref(n_out)))
    return d[:n_out.value].copy(), w[:n_out.value].copy()


class Cloud:
    """Owner of one `pdv_cloud*` (pdv_cloud_create / pdv_cloud_destroy)."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)

    @property
    def handle(self) -> C.c_void_p:
        if not self._h:
            raise ValueError("cloud already destroyed")
        return self._h

    def destroy(self):
        if self._h:
            lib().pdv_cloud_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def info(self) -> dict:
        ci = CloudInfo()
        ci.struct_size = C.sizeof(CloudInfo)
        _check(lib().pdv_cloud_get_info(self.handle, C.byref(ci)))
        return {k: getattr(ci, k) for k, _ in CloudInfo._fields_ if k != "struct_size"}

    def estimated_flights(self, run: dict | None = None) -> float:
        """The library's estimate of the flights per history of this cloud under the run options (pdv_estimated_flights): the
        cost a multi-GPU caller balances its split with."""
        out = C.c_double(0.0)
        o = _opts(dict(n_bins=1, v_lo=0.0, v_hi=1.0, aperture_sr=1.0, **{k: run[k] for k in ("mode", "max_events", "roulette_survival",
                                                                                             "single_scatter_only") if run and k in run}))
        _check(lib().pdv_estimated_flights(self.handle, C.byref(o), C.byref(out)))
        return out.value

    def tables(self) -> dict:
        i = self.info()
        nc, K, nd = i["n_classes"], i["n_phase_bins"], i["n_depth_bins"]
        out = dict(k_ext=np.zeros(nc), k_sca=np.zeros(nc), g=np.zeros(nc), p_class=np.zeros(nc),
                   phase=np.zeros((nc, K + 1)), T_edge=np.zeros(nd + 1))
        _check(lib().pdv_cloud_get_tables(self.handle, *[out[k].ctypes.data for k in
                                                         ("k_ext", "k_sca", "g", "p_class", "phase", "T_edge")]))
        return out

    def image(self) -> dict:
        """The device image of the cloud with its layout (pdv_cloud_get_image): `layout` dict + the sections as numpy views."""
        lay = ImageLayout()
        lay.struct_size = C.sizeof(ImageLayout)
        _check(lib().pdv_cloud_get_image(self.handle, C.byref(lay), None, 0))
        buf = np.zeros(lay.image_bytes, dtype=np.uint8)
        _check(lib().pdv_cloud_get_image(self.handle, C.byref(lay), buf.ctypes.data, buf.size))
        L = {k: getattr(lay, k) for k, _ in ImageLayout._fields_ if k != "struct_size"}
        nct = max(L["n_classes"], 2)
        sec = lambda off, dt, n: np.frombuffer(buf, dtype=dt, count=n, offset=off)
        return dict(layout=L, bytes=buf,
                    phase=sec(L["off_phase"], np.float32, 2 * nct * L["n_phase_bins"]).reshape(nct, L["n_phase_bins"], 2),
                    rows=sec(L["off_rows"], np.float32, 4 * L["n_depth_bins"]).reshape(L["n_depth_bins"], 4),
                    thr=sec(L["off_thr"], np.uint32, PDV_MAX_CLASSES), thr24=sec(L["off_thr24"], np.uint32, PDV_MAX_CLASSES),
                    albedo=sec(L["off_albedo"], np.float32, nct), guide=sec(L["off_guide"], np.uint16, L["n_guide"]),
                    cguide=sec(L["off_cguide"], np.uint8, L["cguide_cells"]))

    def gas_tables(self, t: float) -> dict:
        """Host depth tables of the (cloud, snapshot time t) unit of a cloud in a gas environment (pdv_cloud_gas_tables)."""
        i = self.info()
        nc, nd = i["n_classes"], i["n_depth_bins"]
        out = dict(zeta_edge=np.zeros(nd + 1), T_edge=np.zeros(nd + 1), class_cum=np.zeros((nd, nc)), L=np.zeros(nc))
        _check(lib().pdv_cloud_gas_tables(self.handle, float(t), *[out[k].ctypes.data for k in ("zeta_edge", "T_edge", "class_cum", "L")]))
        return out


def pdv_cloud_create(params: dict) -> Cloud:
    """params: a cloud dictionary as in pdv_workloads._cloud (SI units).  Either explicit `diameters` +
    `number_weights`, or `lognormal={d_median, sigma_ln, n_classes}` (expanded with pdv_lognormal_classes)."""
    if "lognormal" in params:
        ln = params["lognormal"]
        d, w = pdv_lognormal_classes(ln["d_median"], ln["sigma_ln"], ln["n_classes"])
    else:
        d = np.ascontiguousarray(params["diameters"], dtype=np.float64)
        w = np.ascontiguousarray(params["number_weights"], dtype=np.float64)
    dp = C.POINTER(C.c_double)
    p = CloudParams()
    p.struct_size = C.sizeof(CloudParams)
    p.area_mass, p.density, p.v_fs = params["area_mass"], params["density"], params["v_fs"]
    p.profile_kind = int(params.get("profile_kind", 0))
    p.beta, p.vmax_ratio = float(params.get("beta", 0.0)), params["vmax_ratio"]
    keep = [d, w]
    if p.profile_kind == 1:
        pv = np.ascontiguousarray(params["prof_v"], dtype=np.float64)
        pm = np.ascontiguousarray(params["prof_cum_mass"], dtype=np.float64)
        if pv.shape != pm.shape:
            raise ValueError("prof_v / prof_cum_mass shapes differ")
        keep += [pv, pm]
        p.n_prof, p.prof_v, p.prof_cum_mass = pv.size, pv.ctypes.data_as(dp), pm.ctypes.data_as(dp)
    if d.shape != w.shape or d.ndim != 1:
        raise ValueError("diameters / number_weights must be 1-D and of equal length")
    p.n_classes, p.diameter, p.number_weight = d.size, d.ctypes.data_as(dp), w.ctypes.data_as(dp)
    p.m_re, p.m_im, p.wavelength = params["m_re"], params["m_im"], params["wavelength"]
    p.surface_reflectivity, p.surface_model = params["surface_reflectivity"], int(params.get("surface_model", 0))
    p.n_phase_bins, p.n_depth_bins = int(params.get("n_phase_bins", 0)), int(params.get("n_depth_bins", 0))
    p.phase_model = int(params.get("phase_model", 0))
    p.depth_model = int(params.get("depth_model", 0))
    p.gas_density = float(params.get("gas_density", 0.0))
    p.drag_coefficient = float(params.get("drag_coefficient", 0.5 if p.gas_density > 0.0 else 0.0))
    h = C.c_void_p(None)
    _check(lib().pdv_cloud_create(C.byref(p), C.byref(h)))
    return Cloud(h.value)


def _opts(run: dict, output_on_device: bool = False) -> RunOpts:
    o = RunOpts()
    o.struct_size = C.sizeof(RunOpts)
    o.n_bins, o.v_lo, o.v_hi = int(run["n_bins"]), float(run["v_lo"]), float(run["v_hi"])
    o.aperture_sr, o.mode = float(run["aperture_sr"]), int(run.get("mode", 0))
    o.max_events, o.roulette_survival = int(run.get("max_events", 0)), float(run.get("roulette_survival", 0.1))
    o.single_scatter_only = int(run.get("single_scatter_only", 0))
    o.first_photon_id = int(run.get("first_photon_id", 0))
    o.output_on_device = int(output_on_device)
    o.blocks_per_sm, o.threads_per_block = int(run.get("blocks_per_sm", 0)), int(run.get("threads_per_block", 0))
    o.launch_model = int(run.get("launch_model", 0))
    us = run.get("unit_streams")
    if us is not None:                 # [n_clouds * n_snap] sub-stream index of each unit (units of a larger job)
        arr = np.ascontiguousarray(us, dtype=np.uint32)
        o._keep_unit_streams = arr     # keeps the buffer alive as long as the options struct
        o.unit_streams = arr.ctypes.data_as(C.POINTER(C.c_uint32))
    return o


@dataclass
class RunResult:
    hist: np.ndarray          # [n_clouds, n_snap, n_bins]
    hist2: np.ndarray
    stats: np.ndarray         # structured [n_clouds, n_snap], STATS_DTYPE
    n_photons: int

    def conservation_residual(self) -> np.ndarray:
        s = self.stats
        return (s["detected"] + s["underflow"] + s["overflow"] + s["escaped"] + s["absorbed_particles"]
                + s["absorbed_surface"] + s["roulette_killed"] - s["roulette_gained"] + s["truncated"]
                - s["histories"].astype(np.float64))


def pdv_mc_run(clouds, t_snap, n_photons: int, seed: int, run: dict, stream: int | None = None) -> RunResult:
    """Host-buffer call of pdv_mc_run: numpy outputs, returns when they are filled.  `run` holds the run options
    (n_bins, v_lo, v_hi, aperture_sr, mode, max_events, roulette_survival, single_scatter_only, ...)."""
    clouds = list(clouds)
    t = np.ascontiguousarray(t_snap, dtype=np.float64)
    nc, ns, nb = len(clouds), t.size, int(run["n_bins"])
    hist = np.zeros((nc, ns, nb))
    hist2 = np.zeros((nc, ns, nb))
    stats = np.zeros((nc, ns), dtype=STATS_DTYPE)
    arr = (C.c_void_p * nc)(*[c.handle for c in clouds])
    o = _opts(run)
    _check(lib().pdv_mc_run(arr, nc, t.ctypes.data_as(C.POINTER(C.c_double)), ns, int(n_photons), int(seed), C.byref(o),
                            hist.ctypes.data, hist2.ctypes.data, stats.ctypes.data, C.c_void_p(stream)))
    return RunResult(hist, hist2, stats, int(n_photons))


def pdv_mc_run_device(clouds, t_snap, n_photons: int, seed: int, run: dict, hist, hist2=None, stats=None,
                      stream: int | None = None):
    """Device-buffer call: hist/hist2 are CUDA float64 torch tensors [n_clouds, n_snap, n_bins], stats an optional
    CUDA uint8 tensor of n_clouds*n_snap*STATS_DTYPE.itemsize bytes; the call only enqueues work on `stream`
    (default: torch's current stream)."""
    import torch
    clouds = list(clouds)
    t = np.ascontiguousarray(t_snap, dtype=np.float64)
    nc, ns, nb = len(clouds), t.size, int(run["n_bins"])
    for x in (hist, hist2):
        if x is not None and not (x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and x.numel() == nc * ns * nb):
            raise ValueError("hist/hist2 must be contiguous CUDA float64 tensors of n_clouds*n_snap*n_bins elements")
    if stats is not None and not (stats.is_cuda and stats.dtype == torch.uint8 and stats.numel() == nc * ns * STATS_DTYPE.itemsize):
        raise ValueError("stats must be a CUDA uint8 tensor of n_units*STATS_DTYPE.itemsize bytes")
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    arr = (C.c_void_p * nc)(*[c.handle for c in clouds])
    o = _opts(run, output_on_device=True)
    _check(lib().pdv_mc_run(arr, nc, t.ctypes.data_as(C.POINTER(C.c_double)), ns, int(n_photons), int(seed), C.byref(o),
                            hist.data_ptr(), hist2.data_ptr() if hist2 is not None else None,
                            stats.data_ptr() if stats is not None else None, C.c_void_p(stream)))


def pdv_mc_run_static(clouds, t_snap, n_photons: int, seed: int, run: dict, hist, hist2=None, stats=None,
                      stream: int | None = None):
    """pdv_mc_run_device through the entry point that allocates no device memory (pdv_mc_run_static in include/pdv.h).

    For a caller whose process cannot spare the library a device allocation per call -- all HBM already sits in the
    caller's own arena, or the footprint must be fixed when the library is loaded.  The workspace is a fixed 2 MiB array
    inside the library (PDV_STATIC_SCRATCH_BYTES), shared by every call on the device: calls on one stream are safe, calls
    that can overlap on the GPU race.  The clouds must have been created (and so uploaded) beforehand; the tensors are the
    caller's, as for pdv_mc_run_device.  Results are bit-identical to pdv_mc_run_device's.  Raises PdvError
    (PDV_E_UNSUPPORTED) when n_units x n_bins does not fit the array, or for gas clouds."""
    import torch
    clouds = list(clouds)
    t = np.ascontiguousarray(t_snap, dtype=np.float64)
    nc, ns, nb = len(clouds), t.size, int(run["n_bins"])
    for x in (hist, hist2):
        if x is not None and not (x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and x.numel() == nc * ns * nb):
            raise ValueError("hist/hist2 must be contiguous CUDA float64 tensors of n_clouds*n_snap*n_bins elements")
    if stats is not None and not (stats.is_cuda and stats.dtype == torch.uint8 and stats.numel() == nc * ns * STATS_DTYPE.itemsize):
        raise ValueError("stats must be a CUDA uint8 tensor of n_units*STATS_DTYPE.itemsize bytes")
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    arr = (C.c_void_p * nc)(*[c.handle for c in clouds])
    o = _opts(run, output_on_device=True)
    _check(lib().pdv_mc_run_static(arr, nc, t.ctypes.data_as(C.POINTER(C.c_double)), ns, int(n_photons), int(seed), C.byref(o),
                                   hist.data_ptr(), hist2.data_ptr() if hist2 is not None else None,
                                   stats.data_ptr() if stats is not None else None, C.c_void_p(stream)))


def pdv_mc_trace(cloud: Cloud, unit: int, n_photons: int, seed: int, run: dict, stream: int | None = None):
    """-> (RunResult for the single unit, records[n_photons] of TRACE_DTYPE)."""
    nb = int(run["n_bins"])
    hist, hist2 = np.zeros((1, 1, nb)), np.zeros((1, 1, nb))
    stats = np.zeros((1, 1), dtype=STATS_DTYPE)
    rec = np.zeros(int(n_photons), dtype=TRACE_DTYPE)
    o = _opts(run)
    _check(lib().pdv_mc_trace(cloud.handle, int(unit), int(n_photons), int(seed), C.byref(o), hist.ctypes.data,
                              hist2.ctypes.data, stats.ctypes.data, rec.ctypes.data, C.c_void_p(stream)))
    return RunResult(hist, hist2, stats, int(n_photons)), rec


def pdv_spectrogram(hist, n_photons: int, v_lo: float, v_hi: float, scale: int = 0, floor_db: float = -120.0,
                    stream: int | None = None):
    """hist: numpy [n_snap, n_bins] float64 -> numpy float32, or a CUDA float64 torch tensor -> CUDA float32 tensor."""
    if isinstance(hist, np.ndarray):
        h = np.ascontiguousarray(hist, dtype=np.float64)
        if h.ndim != 2:
            raise ValueError("hist must be [n_snap, n_bins]")
        out = np.zeros(h.shape, dtype=np.float32)
        _check(lib().pdv_spectrogram(h.ctypes.data, h.shape[0], h.shape[1], int(n_photons), v_lo, v_hi, scale, floor_db,
                                     out.ctypes.data, 0, C.c_void_p(stream)))
        return out
    import torch
    if not (hist.is_cuda and hist.dtype == torch.float64 and hist.is_contiguous() and hist.dim() == 2):
        raise ValueError("hist must be a contiguous 2-D CUDA float64 tensor")
    out = torch.empty(hist.shape, dtype=torch.float32, device=hist.device)
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    _check(lib().pdv_spectrogram(hist.data_ptr(), hist.shape[0], hist.shape[1], int(n_photons), v_lo, v_hi, scale,
                                 floor_db, out.data_ptr(), 1, C.c_void_p(stream)))
    return out


def pdv_spectrum_peaks(hist, n_photons: int, v_lo: float, v_hi: float, v_fs, *, half: int = 4, n_pass: int = 2,
                       fit_half: int = 8, x_min: float = 1.02, x_max: float = 1e30, stream: int | None = None):
    """Main-peak characteristics (Eq. 35) of each row of hist [n_units, n_bins].

    numpy float64 hist + scalar / array v_fs -> numpy structured array of PEAK_DTYPE;
    CUDA float64 tensors hist [n_units, n_bins] and v_fs [n_units] -> CUDA uint8 tensor of n_units * PEAK_DTYPE.itemsize
    bytes (enqueued on the stream; `.cpu().numpy().view(PEAK_DTYPE)` reads it)."""
    o = PeakOpts(C.sizeof(PeakOpts), int(half), int(n_pass), int(fit_half), 0, float(x_min), float(x_max))
    if isinstance(hist, np.ndarray):
        h = np.ascontiguousarray(hist, dtype=np.float64)
        if h.ndim != 2:
            raise ValueError("hist must be [n_units, n_bins]")
        v = np.ascontiguousarray(np.broadcast_to(np.asarray(v_fs, dtype=np.float64), (h.shape[0],)))
        out = np.zeros(h.shape[0], dtype=PEAK_DTYPE)
        _check(lib().pdv_spectrum_peaks(h.ctypes.data, h.shape[0], h.shape[1], int(n_photons), v_lo, v_hi, v.ctypes.data,
                                        C.byref(o), out.ctypes.data, 0, C.c_void_p(stream)))
        return out
    import torch
    if not (hist.is_cuda and hist.dtype == torch.float64 and hist.is_contiguous() and hist.dim() == 2):
        raise ValueError("hist must be a contiguous 2-D CUDA float64 tensor")
    if not (torch.is_tensor(v_fs) and v_fs.is_cuda and v_fs.dtype == torch.float64 and v_fs.is_contiguous()
            and v_fs.numel() == hist.shape[0]):
        raise ValueError("v_fs must be a contiguous CUDA float64 tensor with one value per row of hist")
    out = torch.empty(hist.shape[0] * PEAK_DTYPE.itemsize, dtype=torch.uint8, device=hist.device)
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    _check(lib().pdv_spectrum_peaks(hist.data_ptr(), hist.shape[0], hist.shape[1], int(n_photons), v_lo, v_hi,
                                    v_fs.data_ptr(), C.byref(o), out.data_ptr(), 1, C.c_void_p(stream)))
    return out


def pdv_phase_sampling_check(cloud: Cloud, class_index: int, n_samples: int, seed: int, n_bins: int = 64,
                             stream: int | None = None) -> dict:
    """cos(theta) of one size class sampled n_samples times from the table and by rejection on the exact Mie function.
    -> dict(hist_table, hist_exact: uint64 [n_bins]; mean_cos_table, mean_cos_exact, i_max, n_trials, n_bound_violations)."""
    ht, he = np.zeros(int(n_bins), dtype=np.uint64), np.zeros(int(n_bins), dtype=np.uint64)
    info = PhaseCheck()
    _check(lib().pdv_phase_sampling_check(cloud.handle, int(class_index), int(n_samples), int(seed), int(n_bins),
                                          ht.ctypes.data, he.ctypes.data, C.byref(info), C.c_void_p(stream)))
    n = max(int(n_samples), 1)
    return dict(hist_table=ht, hist_exact=he, mean_cos_table=info.sum_cos_table / n, mean_cos_exact=info.sum_cos_exact / n,
                i_max=info.i_max, n_trials=int(info.n_trials), n_bound_violations=int(info.n_bound_violations))


def pdv_philox_blocks(counters, seed: int):
    """Raw Philox4x32-10 blocks of the device generator (pdv_philox_blocks): counters uint32 [n, 4], key = the two words of `seed`.
    -> (static, shared, param): uint32 [n, 4] each, one per key path of the transport kernel."""
    c = np.ascontiguousarray(counters, dtype=np.uint32).reshape(-1, 4)
    outs = [np.zeros_like(c) for _ in range(3)]
    _check(lib().pdv_philox_blocks(c.ctypes.data, c.shape[0], int(seed), *[o.ctypes.data for o in outs]))
    return tuple(outs)


def pdv_issue_peaks(millis: float = 50.0, stream: int | None = None) -> dict:
    f, m, z = C.c_double(0), C.c_double(0), C.c_double(0)
    n = C.c_int32(0)
    _check(lib().pdv_issue_peaks(millis, C.byref(f), C.byref(m), C.byref(z), C.byref(n), C.c_void_p(stream)))
    return dict(ffma_thread_inst_per_s=f.value, mufu_thread_inst_per_s=m.value, sm_clock_mhz=z.value, n_sm=n.value)


def pdv_last_launch_info(stream: int | None = None) -> dict:
    """Launch statistics of this thread's last run; stream (a cudaStream_t as int, 0 = the default stream): of its last run on
    that stream (pdv_launch_info_on_stream)."""
    k, g, b, s, v = C.c_int32(0), C.c_int32(0), C.c_int32(0), C.c_int32(0), C.c_int32(0)
    ms = C.c_float(0)
    if stream is None:
        lib().pdv_last_launch_info(C.byref(k), C.byref(ms), C.byref(g), C.byref(b), C.byref(s), C.byref(v))
    else:
        lib().pdv_launch_info_on_stream(C.c_void_p(stream), C.byref(k), C.byref(ms), C.byref(g), C.byref(b), C.byref(s), C.byref(v))
    return dict(n_kernels=k.value, transport_ms=ms.value, grid=g.value, block=b.value, smem_bytes=s.value, variant=v.value,
                alt=bool(v.value & 32))
