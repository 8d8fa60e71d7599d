"""CPU-side checks of the product library: it loads, exports every symbol include/pdv.h declares, validates its
arguments, and its host optics (a second, independent Mie + table implementation in C++) agree with the oracle.
No compute call needs a GPU here; pdv_mc_run must refuse to run without one (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud as ocloud

import paper_2012_00963_b200 as P
from paper_2012_00963_b200 import build as pbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    pbuild.build()


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "pdv.h")).read()
    declared = set(re.findall(r"\b(pdv_[a-z_0-9]+)\s*\(", header))
    declared -= {"pdv_cloud_params", "pdv_run_opts"}
    assert declared == set(P.EXPORTS)
    L = C.CDLL(P.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    assert "sm_100a" in P.pdv_version()


def test_struct_sizes_match_header_layout():
    """The ctypes mirrors must have the C layout: the library checks struct_size."""
    c = P.pdv_cloud_create(W.config(0)["clouds"][0])
    assert c.info()["n_classes"] == 1
    c.destroy()
    with pytest.raises(ValueError):
        c.handle


@pytest.mark.parametrize("idx", [1, 2, 4])
def test_host_optics_match_oracle(idx):
    """Two independent implementations (oracle: scipy Bessel + cumulative Simpson; library: Riccati-Bessel
    recurrences + panel-wise cubic inversion) of Eq. 10, 12-14, 20."""
    params = W.config(idx)["clouds"][0]
    c = P.pdv_cloud_create(params)
    oc = ocloud.build_cloud(params)
    t, i = c.tables(), c.info()
    assert i["tau_ext"] == pytest.approx(oc.tau_ext, rel=1e-12)
    assert i["kappa"] == pytest.approx(oc.kappa, rel=1e-12)
    assert i["sauter_diameter"] == pytest.approx(oc.sauter_diameter, rel=1e-12)
    assert np.allclose(t["k_ext"], oc.k_ext, rtol=1e-11, atol=0)
    assert np.allclose(t["k_sca"], oc.k_sca, rtol=1e-11, atol=0)
    assert np.allclose(t["g"], oc.g, rtol=0, atol=1e-11)
    assert np.allclose(t["p_class"], oc.p_class, rtol=0, atol=1e-13)
    assert np.max(np.abs(t["phase"] - oc.phase)) < 1e-9
    assert np.allclose(t["T_edge"], oc.T_edge, rtol=1e-12, atol=1e-13 * oc.tau_ext)


def test_lognormal_classes_match_oracle():
    for med, sig in ((3e-6, 0.5), (1e-6, 0.7)):
        d, w = P.pdv_lognormal_classes(med, sig, 16)
        do, wo = ocloud.lognormal_classes(med, sig, 16)
        assert np.allclose(d, do, rtol=1e-14) and np.allclose(w, wo, rtol=1e-12, atol=1e-16)
    d, w = P.pdv_lognormal_classes(2e-6, 0.0, 16)
    assert d.tolist() == [2e-6] and w.tolist() == [1.0]


def test_isotropic_phase_model_and_tabulated_profile():
    params = dict(W.config(1)["clouds"][0], phase_model=1)
    c = P.pdv_cloud_create(params)
    t = c.tables()
    assert np.allclose(t["phase"][0], np.linspace(-1, 1, 1025), atol=1e-15) and t["g"][0] == 0.0
    # tabulated profile sampled from the exponential law reproduces the exponential depth table
    base = W.config(1)["clouds"][0]
    v = np.linspace(base["v_fs"], base["vmax_ratio"] * base["v_fs"], 20001)
    cum = 1.0 - np.exp(-base["beta"] * (v / base["v_fs"] - 1.0))
    c1 = P.pdv_cloud_create(dict(base, profile_kind=1, prof_v=v, prof_cum_mass=cum))
    c0 = P.pdv_cloud_create(base)
    assert np.allclose(c1.tables()["T_edge"], c0.tables()["T_edge"], rtol=0, atol=2e-8 * c0.info()["tau_ext"])
    oc = ocloud.build_cloud(dict(base, profile_kind=1, prof_v=v, prof_cum_mass=cum))
    assert np.allclose(c1.tables()["T_edge"], oc.T_edge, rtol=0, atol=1e-12 * oc.tau_ext)


@pytest.mark.parametrize("patch", [dict(area_mass=-1.0), dict(density=0.0), dict(v_fs=0.0), dict(beta=0.0),
                                   dict(vmax_ratio=1.0), dict(surface_reflectivity=1.5), dict(n_phase_bins=1000),
                                   dict(n_depth_bins=5000), dict(wavelength=0.0), dict(m_im=-1.0),
                                   dict(diameters=[0.0], number_weights=[1.0]), dict(surface_model=3), dict(depth_model=2),
                                   dict(depth_model=1, profile_kind=1, prof_v=[2000.0, 6000.0], prof_cum_mass=[0.0, 1.0]),
                                   dict(diameters=[1e-6] * 33, number_weights=[1.0] * 33)])
def test_cloud_create_rejects_invalid(patch):
    with pytest.raises(P.PdvError) as e:
        P.pdv_cloud_create(dict(W.config(0)["clouds"][0], **patch))
    assert e.value.status == 1


def test_run_argument_validation_and_no_cpu_fallback():
    import torch
    cfg = W.config(0)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    for patch in (dict(n_bins=0), dict(n_bins=9000), dict(v_hi=0.0), dict(aperture_sr=0.0), dict(aperture_sr=7.0),
                  dict(mode=2), dict(max_events=-1), dict(max_events=5, roulette_survival=0.0), dict(threads_per_block=100)):
        with pytest.raises(P.PdvError) as e:
            P.pdv_mc_run([c], cfg["t_snap"], 100, 1, dict(cfg["run"], **patch))
        assert e.value.status == 1
    with pytest.raises(P.PdvError) as e:
        P.pdv_mc_run([c], [0.0], 100, 1, cfg["run"])
    assert e.value.status == 1
    with pytest.raises(P.PdvError) as e:                       # exactly 2^33 photons would wrap a 64-bit Q31 tally
        P.pdv_mc_run([c], cfg["t_snap"], 2 ** 33, 1, cfg["run"])
    assert e.value.status == 1 and "2^33" in str(e.value)
    if not torch.cuda.is_available():
        with pytest.raises(P.PdvError) as e:
            P.pdv_mc_run([c], cfg["t_snap"], 100, 1, cfg["run"])
        assert e.value.status == 3 and "no CPU fallback" in str(e.value)
        with pytest.raises(P.PdvError):
            P.pdv_spectrogram(np.ones((2, 4)), 10, 0.0, 1.0)
        with pytest.raises(P.PdvError) as e:
            P.pdv_spectrum_peaks(np.ones((2, 64)), 10, 0.0, 6000.0, 2000.0)
        assert e.value.status == 3 and "no CPU fallback" in str(e.value)
    for args in ((1, 10, 1, 8), (0, 10, 1, 0), (0, 10, 1, 5000)):                                   # class / n_bins out of range
        with pytest.raises(P.PdvError) as e:
            P.pdv_phase_sampling_check(c, *args)
        assert e.value.status == 1
    if not torch.cuda.is_available():
        with pytest.raises(P.PdvError) as e:
            P.pdv_phase_sampling_check(c, 0, 10, 1, 8)
        assert e.value.status == 3
    for bad in (dict(half=-1), dict(n_pass=17), dict(fit_half=0), dict(x_min=2.0, x_max=1.0)):      # rejected before any CUDA call
        with pytest.raises(P.PdvError) as e:
            P.pdv_spectrum_peaks(np.ones((2, 64)), 10, 0.0, 6000.0, 2000.0, **bad)
        assert e.value.status == 1
    with pytest.raises(P.PdvError) as e:
        P.pdv_spectrum_peaks(np.ones((2, 64)), 10, 0.0, 6000.0, [2000.0, 0.0])
    assert e.value.status == 1
    assert len(P.pdv_spectrum_peaks(np.ones((0, 64)), 10, 0.0, 6000.0, 2000.0)) == 0                 # n_units = 0 is valid


def test_static_scratch_entry_validates_before_any_cuda_call():
    """pdv_mc_run_static (the entry point that allocates no device memory): host outputs are refused, and without a device it
    reports PDV_E_CUDA like pdv_mc_run.  Through raw ctypes: the Python wrapper wants CUDA tensors."""
    import torch
    from paper_2012_00963_b200 import _binding as B
    cfg = W.config(0)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    L = P.lib()
    arr = (C.c_void_p * 1)(c.handle)
    t = np.asarray(cfg["t_snap"], dtype=np.float64)
    dummy = np.zeros(cfg["run"]["n_bins"])                      # never written: every call below fails first
    call = lambda o, n_snap=1: L.pdv_mc_run_static(arr, 1, t.ctypes.data_as(C.POINTER(C.c_double)), n_snap, 100, 1, C.byref(o),
                                                   dummy.ctypes.data, None, None, None)
    assert call(B._opts(cfg["run"], output_on_device=False)) == 1 and "output_on_device" in L.pdv_last_error().decode()
    assert call(B._opts(dict(cfg["run"], n_bins=0), output_on_device=True)) == 1
    assert call(B._opts(cfg["run"], output_on_device=True), n_snap=0) == 1
    if not torch.cuda.is_available():
        assert call(B._opts(cfg["run"], output_on_device=True)) == 3 and "no CPU fallback" in L.pdv_last_error().decode()
    assert not dummy.any()


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2012_00963_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h", ".hpp", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "pdv_oracle" not in src and "oracle/" not in src.replace("shares nothing with oracle/", ""), f


@pytest.mark.parametrize("idx,n_depth", [(1, 1024), (2, 256)])
def test_host_gas_tables_agree_with_the_oracle(idx, n_depth):
    """Row f4 (R35-R37): the product's per-snapshot depth tables of a cloud in a gas environment (C++,
    csrc/pdv_optics.cpp::build_gas_unit) against the oracle's (numpy, oracle/gas.py) -- two implementations of the same
    reading, no shared code.  No GPU needed."""
    from oracle import gas as ogas
    params = dict(W.config(idx)["clouds"][0], gas_density=5.0, drag_coefficient=0.5, n_depth_bins=n_depth)
    c = P.pdv_cloud_create(params)
    oc = ocloud.build_cloud(params)
    for t in (0.7e-6, 9e-6):
        a, b = c.gas_tables(t), ogas.build_tables(oc, params, t, n_depth)
        assert np.allclose(a["zeta_edge"], b["zeta_edge"], rtol=1e-12, atol=1e-15 * b["zeta_edge"][0])
        assert np.allclose(a["T_edge"], b["T_edge"], rtol=0, atol=1e-12 * oc.tau_ext)
        assert np.allclose(a["class_cum"], b["class_cum"], rtol=0, atol=1e-9)
        assert np.allclose(a["L"], b["L"], rtol=1e-14)
    with pytest.raises(P.PdvError):                      # a vacuum cloud has no per-snapshot tables
        P.pdv_cloud_create(W.config(idx)["clouds"][0]).gas_tables(1e-6)
