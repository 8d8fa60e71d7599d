"""GPU: the paper's own scattering-angle sampler (acceptance-rejection on the exact Mie function, step (4))
on the device, against the table sampler of the hot path and against oracle/phase_check.py.

Counts are binomial: every bin must sit within 5 sigma of N p_j with p_j from the oracle -- exact_bin_probabilities for the
rejection sampler, table_bin_probabilities of the ORACLE's own D_K for the table sampler -- and chi^2 over the bins must be
ordinary.  Means: <cos theta> -> g of the Mie series.  Acceptance: n_samples / n_trials -> int I dmu / (2 i_max).
"""
import math

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud as ocloud, mie as omie, phase_check as opc

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("_library_is_built")]
M_SN = complex(W.M_RE, W.M_IM)


def _binomial_check(counts, p, n):
    counts = np.asarray(counts, dtype=np.float64)
    assert counts.sum() == n
    sig = np.sqrt(np.maximum(n * p * (1 - p), 1.0))
    z = (counts - n * p) / sig
    assert np.max(np.abs(z)) < 5.0, (np.argmax(np.abs(z)), z[np.argmax(np.abs(z))])
    chi2 = float(np.sum(z ** 2))
    assert chi2 < len(p) + 6 * math.sqrt(2 * len(p)) + 10, chi2


@pytest.mark.parametrize("d_um,n_bins", [(5.0, 64), (1.0, 200), (10.0, 33)])
def test_both_samplers_match_their_expected_histograms(d_um, n_bins):
    import paper_2012_00963_b200 as P
    params = W._cloud(2.0, 4.0, 2000.0, diameter_um=d_um)
    c = P.pdv_cloud_create(params)
    n = 4_000_000
    r = P.pdv_phase_sampling_check(c, 0, n, 123, n_bins)
    x = math.pi * d_um * 1e-6 / W.WAVELENGTH
    assert r["n_bound_violations"] == 0
    _binomial_check(r["hist_exact"], opc.exact_bin_probabilities(x, M_SN, n_bins), n)
    _binomial_check(r["hist_table"], opc.table_bin_probabilities(ocloud.phase_quantile_table(x, M_SN, 1024), n_bins), n)
    g = omie.efficiencies(x, M_SN)[3]
    # variance of cos(theta) is below 1: 5 sigma of the mean is 5 / sqrt(n)
    assert r["mean_cos_exact"] == pytest.approx(g, abs=5 / math.sqrt(n))
    assert r["mean_cos_table"] == pytest.approx(g, abs=5 / math.sqrt(n))
    total, imax = opc.intensity_integral_and_max(x, M_SN)
    assert r["i_max"] == pytest.approx(1.02 * imax, rel=1e-3)              # the host's bound: grid maximum + 2 %
    acc = n / r["n_trials"]
    want = total / (2 * r["i_max"])
    assert acc == pytest.approx(want, rel=5 * math.sqrt((1 - want) / (want * r["n_trials"])) + 1e-4)
    # the table error the check is there to report: total variation between the two device histograms is sampling noise
    tv = opc.total_variation(r["hist_table"], r["hist_exact"])
    assert tv < 3 * math.sqrt(n_bins / n)


def test_polydisperse_classes_reproducibility_and_arguments():
    import paper_2012_00963_b200 as P
    cfg = W.config(2)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    info = c.info()
    n = 500_000
    for cls in (0, 7, 15):
        r = P.pdv_phase_sampling_check(c, cls, n, 5, 50)
        r2 = P.pdv_phase_sampling_check(c, cls, n, 5, 50)
        assert np.array_equal(r["hist_exact"], r2["hist_exact"]) and np.array_equal(r["hist_table"], r2["hist_table"])
        assert r["n_trials"] == r2["n_trials"] and r["n_bound_violations"] == 0
        assert r["hist_exact"].sum() == n and r["hist_table"].sum() == n
        assert r["mean_cos_exact"] == pytest.approx(r["mean_cos_table"], abs=7 / math.sqrt(n))
        assert opc.total_variation(r["hist_table"], r["hist_exact"]) < 3 * math.sqrt(50 / n)
    assert info["n_classes"] == 16
    z = P.pdv_phase_sampling_check(c, 0, 0, 1, 8)
    assert z["hist_exact"].sum() == 0 and z["n_trials"] == 0
    one = P.pdv_phase_sampling_check(c, 3, 1, 1, 1)                          # one sample, one bin
    assert one["hist_exact"][0] == 1 and one["hist_table"][0] == 1
    for bad in (dict(class_index=16), dict(class_index=-1), dict(n_bins=0), dict(n_bins=5000)):
        kw = dict(class_index=0, n_samples=10, seed=1, n_bins=8)
        kw.update(bad)
        with pytest.raises(P.PdvError) as e:
            P.pdv_phase_sampling_check(c, kw["class_index"], kw["n_samples"], kw["seed"], kw["n_bins"])
        assert e.value.status == 1
    iso = P.pdv_cloud_create(dict(W.config(1)["clouds"][0], phase_model=1))
    with pytest.raises(P.PdvError) as e:
        P.pdv_phase_sampling_check(iso, 0, 10, 1, 8)
    assert e.value.status == 4
