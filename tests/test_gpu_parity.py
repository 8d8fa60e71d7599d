"""GPU parity tests: the CUDA path (through the C-ABI) against the fp64 CPU oracle on the same seeded inputs.

The method is a stochastic estimator, so parity is statistical (north_star): per (merged) bin
|gpu - cpu| <= 5 sqrt(var_gpu + var_cpu), plus 1e-3 relative on the weight leaving the cloud top at >= 1e8
photons (reading R22).  Where both sides can run the SAME counter-based random stream (oracle
rng_mode 1 = DESIGN.md D1/D2) single histories are compared one by one.  Integer work (tallies, counters,
conservation, determinism) is bit-exact.
"""
import math

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud as ocloud
from oracle import mc as omc

from histcmp import compare, load_golden, per_history_variance

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("_library_is_built")]


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2012_00963_b200 import build as pbuild
    pbuild.build()
    import paper_2012_00963_b200 as P
    return P


def _oracle(params, run, n, **kw):
    oc = ocloud.build_cloud(params)
    return omc.run(oc, dict(run, seed=987654321), n_photons=n, **kw)


def _assert_hist_parity(g_hist, g_hist2, n_g, o, min_ndf=5, min_eff=25.0):
    res = compare(g_hist, g_hist2, n_g, o.hist, o.hist2, o.n_photons, min_eff=min_eff)
    assert res["ndf"] >= min_ndf
    assert res["worst"] < 5.0, res["z"]
    assert res["chi2"] < res["ndf"] + 6 * math.sqrt(2 * res["ndf"]) + 10
    return res


def _assert_stats_parity(gs, n_g, o, same_game=True):
    """Weights leaving / absorbed per photon agree within 5 sigma of a conservative variance bound (w <= 1).
    same_game=False: the two sides play Russian roulette under different rules (the kernel only while w/p <= 1,
    DESIGN.md reading R20), so the number of events per history is not comparable, only the expectations are."""
    for key in ("detected", "escaped", "absorbed_particles", "absorbed_surface", "truncated"):
        a, b = float(gs[key]) / n_g, o.stats[key] / o.n_photons
        sig = math.sqrt(max(a, 1e-12) / n_g + max(b, 1e-12) / o.n_photons)      # Bernoulli bound: w <= 1 gives var <= mean
        # A history's share of `absorbed_particles` or `escaped` is far from 0/1, so that bound is 2-3 times too wide for them.
        # Stored oracle runs carry per-chunk statistics: the batch-means variance of one history's contribution (both sides
        # sample the same distribution, so it serves the GPU's term too), times 1.5 for the uncertainty of that estimate.
        var_h = per_history_variance(o, key) if hasattr(o, "chunk_stats") else None
        if var_h is not None:
            sig = min(sig, 1.5 * math.sqrt(var_h / n_g + var_h / o.n_photons) + 1e-15)
        assert abs(a - b) < 5 * sig, (key, a, b, sig)
    if same_game:
        a = float(gs["particle_events"]) / n_g
        b = o.stats["particle_events"] / o.n_photons
        assert a == pytest.approx(b, rel=0.02)


# -------------------------------------------------------------------------------------------------- configs
def test_config1_exact_size(P):
    """BASELINE.json configs[0] as specified: 1e5 photons, seed 1, 512 bins (oracle at 2e6 for a sharper reference)."""
    cfg = W.config(0)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = cfg["run"]["n_photons"]
    r = P.pdv_mc_run([c], cfg["t_snap"], n, cfg["run"]["seed"], cfg["run"])
    o = _oracle(cfg["clouds"][0], cfg["run"], 2_000_000)
    _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, o, min_ndf=3)
    _assert_stats_parity(r.stats[0, 0], n, o)
    assert r.stats[0, 0]["histories"] == n and r.conservation_residual()[0, 0] == 0.0


def test_config2_scaled(P):
    cfg = W.config(1)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = 4_000_037                                   # ragged: not a multiple of 32 or of the chunk
    r = P.pdv_mc_run([c], cfg["t_snap"], n, 2, cfg["run"])
    o = _oracle(cfg["clouds"][0], cfg["run"], 4_000_000)
    res = _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, o, min_ndf=100)
    _assert_stats_parity(r.stats[0, 0], n, o)
    assert r.stats[0, 0]["histories"] == n
    assert int(r.stats[0, 0]["max_events_in_history"]) > 40
    assert np.argmax(r.hist[0, 0]) == np.argmax(o.hist)          # free-surface peak bin (just below v_fs)


def test_config3_polydisperse_multi_snapshot(P):
    """16 size classes, 6 snapshots in one launch; every row matches the oracle and rows are mutually consistent
    (time invariance in vacuum, reading R16 / pin P10)."""
    cfg = W.scaled(W.config(2), 600_000, n_snap=6)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = cfg["run"]["n_photons"]
    r = P.pdv_mc_run([c], cfg["t_snap"], n, 3, cfg["run"])
    o = _oracle(cfg["clouds"][0], cfg["run"], 2_000_000)
    for i in range(6):
        _assert_hist_parity(r.hist[0, i], r.hist2[0, i], n, o, min_ndf=30)
        assert r.stats[0, i]["histories"] == n
    assert not np.array_equal(r.hist[0, 0], r.hist[0, 1])       # independent random streams per unit
    _assert_stats_parity({k: r.stats[0][k].sum() for k in r.stats.dtype.names}, 6 * n, o)
    res = compare(r.hist[0, 0], r.hist2[0, 0], n, r.hist[0, 5], r.hist2[0, 5], n)
    assert res["worst"] < 5.0


def test_config4_sweep_subset(P):
    """Heterogeneous clouds in one launch: thin/thick, small/large particles, both betas."""
    cfg = W.config(3)
    pick = [0, 7, 17, 30, 41, 47]
    params = [cfg["clouds"][i] for i in pick]
    clouds = [P.pdv_cloud_create(p) for p in params]
    n = 300_000
    r = P.pdv_mc_run(clouds, cfg["t_snap"], n, 4, cfg["run"])
    for i, p in enumerate(params):
        o = _oracle(p, cfg["run"], 300_000)
        _assert_hist_parity(r.hist[i, 0], r.hist2[i, 0], n, o, min_ndf=5)
        _assert_stats_parity(r.stats[i, 0], n, o)
        assert r.stats[i, 0]["histories"] == n and r.conservation_residual()[i, 0] == 0.0


def test_config5_thick_roulette_scaled(P):
    cfg = W.config(4)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = 400_000
    r = P.pdv_mc_run([c], cfg["t_snap"], n, 5, cfg["run"])
    o = _oracle(cfg["clouds"][0], cfg["run"], 400_000)
    _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, o, min_ndf=50)
    _assert_stats_parity(r.stats[0, 0], n, o)
    s = r.stats[0, 0]
    assert s["max_events_in_history"] >= 200 and s["roulette_killed"] > 0
    assert r.conservation_residual()[0, 0] == 0.0


# -------------------------------------------------------------------------------------------------- same random stream
@pytest.mark.parametrize("idx,mode", [(1, 0), (1, 1), (2, 0)])
def test_history_by_history_on_shared_philox_stream(P, idx, mode):
    """Both sides implement the counter-based stream of DESIGN.md D1/D2, so history i makes the same decisions on
    both; fp32 vs fp64 rounding can flip a branch only at a boundary (rare) and moves v~ by rounding only."""
    cfg = W.config(idx)
    run = dict(cfg["run"], mode=mode)
    params = cfg["clouds"][0]
    c = P.pdv_cloud_create(params)
    n, seed, unit = 200_000, 424242, 3
    r, rec = P.pdv_mc_trace(c, unit, n, seed, run)
    oc = ocloud.build_cloud(params)
    o = omc.run(oc, dict(run, seed=seed), n_photons=n, rng_mode=1, stream=unit, trace=True)
    tr = o.trace
    g_fate = np.where(rec["fate"] == 5, 0, rec["fate"])
    same = (g_fate == tr["fate"]) & (rec["n_scatter"] == tr["n_scatter"]) & (rec["n_reflect"] == tr["n_reflect"])
    if mode == 0:
        # the weight is the product of the albedos of the classes that were hit: a different weight = a different class
        # somewhere (the two sides' cumulative class probabilities agree to 1e-9, i.e. a few units of the 32-bit class
        # word: about one pick in 1e8 falls between them)
        same &= np.abs(rec["weight"] - tr["w"]) < 1e-6
    assert same.mean() > 0.999, same.mean()
    out = same & (tr["fate"] <= 1)
    assert out.sum() > 0.3 * n
    dv = np.abs(rec["vt"][out] - tr["vt"][out])
    # fp32 tolerance ("History by history"): one event moves v~ by 1/2 v dmu with dmu ~ 1e-6 (cos.approx
    # 2^-21.4 abs, sqrt.approx, lg2.approx, fma rounding) => ~3e-3 m/s per event at v ~ 6 km/s, a random walk over the ~10-20
    # events of a history.  The same dmu shifts the end of the next flight by dT ~ 1e-6, and where v(T) is logarithmic (the
    # top 3e-4 of the optical depth: dv/dT ~ 8e5 m/s) that is ~1 m/s: a few histories in 1e5 scatter there.  Bins are
    # 11.7 m/s wide.  Measured at this size (profiles/README.md, round 2): median 1.5e-4 ... 2.7e-4, 99.9 % 0.03 ... 0.09,
    # max 0.5 ... 2.5 m/s, max |d mu_exit| 6e-5 ... 2.8e-4.  max < 20 m/s and max |d mu_exit| < 1e-3 are the bounds the test
    # was introduced with; the 99.9 % quantile was 0.05 for the first kernel (libm logf / sincosf) and is 0.15 since the
    # kernel evaluates ln, cos and sqrt on the SFU (__cosf in commit a2d46aa; the bound was widened in 6a5f781).
    assert np.median(dv) < 0.005 and np.quantile(dv, 0.999) < 0.15 and np.mean(dv > 1.0) < 1e-4 and dv.max() < 20.0
    dmu = np.abs(rec["mu_exit"][out] - tr["mu_exit"][out])
    assert dmu.max() < 1e-3
    # identical decisions => near-identical histograms, far tighter than the statistical tolerance
    assert abs(r.hist.sum() - o.hist.sum()) < 2e-3 * o.hist.sum() + 5
    assert np.sum(np.abs(r.hist[0, 0] - o.hist)) < 0.01 * o.hist.sum() + 10
    assert int(r.stats[0, 0]["particle_events"]) == pytest.approx(o.stats["particle_events"], rel=2e-3)


# -------------------------------------------------------------------------------------------------- integer exactness
def test_bit_identical_for_any_launch_shape_and_id_split(P):
    cfg = W.scaled(W.config(2), 150_001, n_snap=2)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = cfg["run"]["n_photons"]
    a = P.pdv_mc_run([c], cfg["t_snap"], n, 11, cfg["run"])
    b = P.pdv_mc_run([c], cfg["t_snap"], n, 11, dict(cfg["run"], blocks_per_sm=1, threads_per_block=96))
    assert np.array_equal(a.hist, b.hist) and np.array_equal(a.hist2, b.hist2)
    for k in a.stats.dtype.names:
        assert np.array_equal(a.stats[k], b.stats[k]), k
    h1 = P.pdv_mc_run([c], cfg["t_snap"], 70_000, 11, cfg["run"])
    h2 = P.pdv_mc_run([c], cfg["t_snap"], n - 70_000, 11, dict(cfg["run"], first_photon_id=70_000))
    assert np.array_equal(a.hist, h1.hist + h2.hist)
    assert np.array_equal(a.stats["particle_events"], h1.stats["particle_events"] + h2.stats["particle_events"])
    assert np.array_equal(a.stats["escaped"], h1.stats["escaped"] + h2.stats["escaped"])
    other = P.pdv_mc_run([c], cfg["t_snap"], n, 12, cfg["run"])
    assert not np.array_equal(a.hist, other.hist)


@pytest.mark.parametrize("kw", [dict(), dict(mode=1), dict(single_scatter_only=1), dict(max_events=3, roulette_survival=0.5),
                                dict(mode=1, max_events=2, roulette_survival=0.3)])
def test_weight_conservation_is_exact_in_fixed_point(P, kw):
    cfg = W.config(1)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = 500_000
    r = P.pdv_mc_run([c], cfg["t_snap"], n, 21, dict(cfg["run"], **kw))
    assert r.conservation_residual()[0, 0] == 0.0
    assert r.hist.sum() == r.stats[0, 0]["detected"]
    if kw.get("mode") == 1 and not kw.get("max_events"):
        assert np.array_equal(r.hist, r.hist2)                   # analog: every weight is exactly 1
        assert np.all(r.hist == np.round(r.hist))


# -------------------------------------------------------------------------------------------------- variants, edge cases
@pytest.mark.parametrize("kw,ckw", [(dict(mode=1), dict()), (dict(single_scatter_only=1), dict()),
                                    (dict(), dict(surface_model=1)), (dict(), dict(phase_model=1)),
                                    (dict(max_events=6, roulette_survival=0.8), dict()),
                                    (dict(n_bins=8192, v_lo=1000.0, v_hi=5000.0), dict(surface_reflectivity=1.0)),
                                    (dict(aperture_sr=2 * math.pi), dict(surface_reflectivity=0.0)),
                                    # conservative scattering (real index: albedo 1), lossless Lambertian bottom: the cloud of pin P16
                                    (dict(v_lo=-6000.0, v_hi=12000.0), dict(m_re=1.5, m_im=0.0, surface_model=1, surface_reflectivity=1.0))])
def test_variants_match_oracle(P, kw, ckw):
    cfg = W.config(1)
    params = dict(cfg["clouds"][0], **ckw)
    run = dict(cfg["run"], **kw)
    c = P.pdv_cloud_create(params)
    n = 1_000_000
    r = P.pdv_mc_run([c], cfg["t_snap"], n, 31, run)
    if ckw.get("phase_model") == 1:
        oc = ocloud.build_cloud(params, phase_override=ocloud.isotropic_quantile_table(1024)[None, :])
        o = omc.run(oc, dict(run, seed=5), n_photons=n)
    else:
        o = _oracle(params, run, n)
    _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, o, min_ndf=3)
    _assert_stats_parity(r.stats[0, 0], n, o, same_game="max_events" not in kw)
    for key in ("underflow", "overflow"):
        a, b = float(r.stats[0, 0][key]) / n, o.stats[key] / n
        assert abs(a - b) < 5 * math.sqrt((a + b + 1e-9) / n)


def test_tabulated_profile_matches_oracle(P):
    """profile_kind 1: a two-slope mass profile with an empty velocity gap (zero-width depth bins)."""
    base = W.config(1)["clouds"][0]
    v = np.array([2000.0, 2600.0, 3400.0, 3400.001, 6000.0])
    cum = np.array([0.0, 0.7, 0.7, 0.7, 1.0])
    params = dict(base, profile_kind=1, prof_v=v, prof_cum_mass=cum)
    c = P.pdv_cloud_create(params)
    n = 1_000_000
    run = W.config(1)["run"]
    r = P.pdv_mc_run([c], [1e-6], n, 41, run)
    o = _oracle(params, run, n)
    _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, o, min_ndf=50)
    _assert_stats_parity(r.stats[0, 0], n, o)


@pytest.mark.parametrize("idx", [1, 2])
def test_closed_form_depth_model_matches_oracle_and_the_table(P, idx):
    """depth_model 1 (v(T) from the closed form of the truncated Eq. 20, R26) against
    the oracle's analytic-profile variant, and history by history against the depth table on the same Philox stream:
    the 1024-bin table is linear in v inside a bin, so the two velocities differ by < 0.01 m/s per event."""
    cfg = W.config(idx)
    params = dict(cfg["clouds"][0], depth_model=1)
    run = cfg["run"]
    c1 = P.pdv_cloud_create(params)
    c0 = P.pdv_cloud_create(cfg["clouds"][0])
    n = 1_000_000
    r = P.pdv_mc_run([c1], cfg["t_snap"][:1], n, 53, run)
    assert r.conservation_residual()[0, 0] == 0.0
    o = _oracle(cfg["clouds"][0], run, n, analytic_profile=True)
    _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, o, min_ndf=30)
    _assert_stats_parity(r.stats[0, 0], n, o)
    m = 200_000
    _, ta = P.pdv_mc_trace(c1, 0, m, 77, run)
    _, tb = P.pdv_mc_trace(c0, 0, m, 77, run)
    same = (ta["fate"] == tb["fate"]) & (ta["n_scatter"] == tb["n_scatter"]) & (ta["n_reflect"] == tb["n_reflect"])
    assert same.mean() == 1.0                       # the velocity does not steer a history: identical decisions
    dv = np.abs(ta["vt"].astype(np.float64) - tb["vt"].astype(np.float64))
    assert np.median(dv) < 0.02 and np.quantile(dv, 0.999) < 0.5
    # empty cloud: every event is at the surface, v = v_fs exactly
    ce = P.pdv_cloud_create(dict(params, area_mass=0.0))
    re_ = P.pdv_mc_run([ce], cfg["t_snap"][:1], 100_000, 7, run)
    rt = P.pdv_mc_run([P.pdv_cloud_create(dict(cfg["clouds"][0], area_mass=0.0))], cfg["t_snap"][:1], 100_000, 7, run)
    assert np.array_equal(re_.hist, rt.hist)
    with pytest.raises(P.PdvError):                 # the closed form exists for the exponential profile only
        P.pdv_cloud_create(dict(params, profile_kind=1, prof_v=np.array([2000.0, 6000.0]), prof_cum_mass=np.array([0.0, 1.0])))


def test_empty_and_tiny_runs_and_empty_cloud(P):
    cfg = W.config(1)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    r = P.pdv_mc_run([c], cfg["t_snap"], 0, 1, cfg["run"])
    assert r.hist.sum() == 0 and r.stats[0, 0]["histories"] == 0
    for n in (1, 31, 33):
        r = P.pdv_mc_run([c], cfg["t_snap"], n, 1, cfg["run"])
        assert r.stats[0, 0]["histories"] == n and r.conservation_residual()[0, 0] == 0.0
    # no ejecta at all: every photon reflects once off the free surface; detected fraction = R * 0.1137 (pin P9)
    c0 = P.pdv_cloud_create(dict(cfg["clouds"][0], area_mass=0.0))
    n = 1_000_000
    r = P.pdv_mc_run([c0], cfg["t_snap"], n, 7, cfg["run"])
    s = r.stats[0, 0]
    assert s["particle_events"] == 0 and s["surface_reflections"] == n
    frac = math.acos(1 - 0.1 / (2 * math.pi)) / (math.pi / 2)
    assert s["detected"] / n == pytest.approx(0.6 * frac, abs=5 * math.sqrt(0.6 * frac / n))
    assert s["absorbed_surface"] / n == pytest.approx(0.4, abs=1e-6)
    k_lo, k_hi = int(0.5 * (2 - 0.1 / (2 * math.pi)) * 2000 / (6000 / 512)), int(2000 / (6000 / 512))
    assert r.hist[0, 0, k_lo:k_hi + 1].sum() == s["detected"]


def test_closed_form_backscatter_histogram_on_gpu(P):
    """Pins P1 / P9 evaluated on the GPU itself, two-sided, with no reference implementation in the loop: tin spheres of
    50 nm are almost pure absorbers at 1550 nm (x = 0.1: K_sca ~ x^4, K_abs ~ x, albedo 0.024), so the weight in the bins
    just below v_fs is the direct surface reflection alone,
        N e^-tau R (2/pi) int_0^{acos mu_a} exp(-tau / cos th) dth        (Beer-Lambert Eq. 7/10 down and up),
    and photons that also scattered once near the surface add less than 1e-3 of it."""
    cfg = W.config(0)
    params = dict(cfg["clouds"][0], diameters=[0.05e-6], area_mass=1.0 * W.MG_CM2)
    c = P.pdv_cloud_create(params)
    info = c.info()
    tau = info["tau_ext"]
    assert 0.4 < tau < 2.0 and info["mean_albedo"] < 0.03
    n = 8_000_000
    th = (np.arange(20000) + 0.5) / 20000 * math.acos(1 - 0.1 / (2 * math.pi))
    p_direct = math.exp(-tau) * 0.6 * (2 / math.pi) * np.sum(np.exp(-tau / np.cos(th))) * (th[1] - th[0])
    dv = 6000 / 512
    k_lo, k_hi = int(0.5 * (2 - 0.1 / (2 * math.pi)) * 2000 / dv), int(2000 / dv)
    for mode in (0, 1):                             # implicit capture (weights 0.6) and analog (weights 1)
        r = P.pdv_mc_run([c], cfg["t_snap"], n, 3 + mode, dict(cfg["run"], mode=mode))
        s = r.stats[0, 0]
        direct = r.hist[0, 0, k_lo:k_hi + 1].sum()
        var = r.hist2[0, 0, k_lo:k_hi + 1].sum()
        assert abs(direct - n * p_direct) < 5 * math.sqrt(var) + 1e-3 * n * p_direct, (mode, direct, n * p_direct)
        # photons that reach the surface unscattered ~ Binomial(n, e^-tau) and leave (1 - R) of their weight there; the few
        # that scattered first (albedo 0.024) add less than 1 %
        assert float(s["absorbed_surface"]) == pytest.approx(0.4 * n * math.exp(-tau), rel=0.02)
        assert r.conservation_residual()[0, 0] == 0.0


# -------------------------------------------------------------------------------------------------- outputs
def test_device_output_path_and_spectrogram(P):
    import torch
    cfg = W.scaled(W.config(2), 200_000, n_snap=3)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n, nb = cfg["run"]["n_photons"], cfg["run"]["n_bins"]
    host = P.pdv_mc_run([c], cfg["t_snap"], n, 9, cfg["run"])
    hist = torch.zeros((1, 3, nb), dtype=torch.float64, device="cuda")
    hist2 = torch.zeros_like(hist)
    stats = torch.zeros(3 * P.STATS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        P.pdv_mc_run_device([c], cfg["t_snap"], n, 9, cfg["run"], hist, hist2, stats)
        spec = P.pdv_spectrogram(hist[0], n, 0.0, 6000.0, scale=2, floor_db=-90.0)
    st.synchronize()
    assert np.array_equal(hist.cpu().numpy(), host.hist) and np.array_equal(hist2.cpu().numpy(), host.hist2)
    ds = np.frombuffer(stats.cpu().numpy().tobytes(), dtype=P.STATS_DTYPE)
    for k in ds.dtype.names:
        assert np.array_equal(ds[k], host.stats[0][k]), k
    ref = np.where(host.hist[0] > 0, np.maximum(10 * np.log10(np.maximum(host.hist[0], 1e-300) / n), -90.0), -90.0)
    assert np.allclose(spec.cpu().numpy(), ref, atol=2e-4)
    lin = P.pdv_spectrogram(host.hist[0], n, 0.0, 6000.0, scale=0)
    den = P.pdv_spectrogram(host.hist[0], n, 0.0, 6000.0, scale=1)
    assert np.allclose(lin, host.hist[0] / n, rtol=1e-6) and np.allclose(den, host.hist[0] / n / (6000.0 / nb), rtol=1e-6)
    assert lin.shape == (3, nb) and lin.dtype == np.float32


def test_two_device_output_runs_on_two_streams_are_independent(P):
    """Two output_on_device = 1 runs with different n_bins enqueued back to back on two streams from one host thread (the
    second needs the larger scratch): each must equal its host-buffer twin bit for bit.  The device scratch of a call is
    stream-ordered (include/pdv.h, "Streams"), so neither run can zero, reuse or free what the other is using."""
    import torch
    cfg = W.scaled(W.config(1), 3_000_000)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = cfg["run"]["n_photons"]
    runs = [dict(cfg["run"], n_bins=256), dict(cfg["run"], n_bins=8192, v_lo=500.0, v_hi=5500.0)]
    seeds = [101, 202]
    twins = [P.pdv_mc_run([c], cfg["t_snap"], n, sd, r) for sd, r in zip(seeds, runs)]
    for rep in range(3):
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        outs = [(torch.zeros((1, 1, r["n_bins"]), dtype=torch.float64, device="cuda"),
                 torch.zeros((1, 1, r["n_bins"]), dtype=torch.float64, device="cuda"),
                 torch.zeros(P.STATS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")) for r in runs]
        torch.cuda.synchronize()
        for sd, r, st, (h, h2, stt) in zip(seeds, runs, streams, outs):       # back to back: both kernels are in flight together
            P.pdv_mc_run_device([c], cfg["t_snap"], n, sd, r, h, h2, stt, stream=st.cuda_stream)
        torch.cuda.synchronize()
        for (h, h2, stt), tw in zip(outs, twins):
            assert np.array_equal(h.cpu().numpy(), tw.hist) and np.array_equal(h2.cpu().numpy(), tw.hist2)
            ds = np.frombuffer(stt.cpu().numpy().tobytes(), dtype=P.STATS_DTYPE)
            for k in ds.dtype.names:
                assert np.array_equal(ds[k], tw.stats[0][k]), k


@pytest.mark.parametrize("idx,n_snap,n_clouds,scaling", [(1, None, None, "strong"), (2, 5, None, "strong"), (3, None, 6, "strong"),
                                                         (1, None, None, "weak")])
def test_sharded_runs_reduce_to_the_single_run_bit_for_bit(P, idx, n_snap, n_clouds, scaling):
    """SURVEY.md 8(e) on one GPU: the shares of a 3-rank job (paper_2012_00963_b200/_shard.py::plan, what bench.py --gpus N runs:
    id ranges for one unit, whole units -- with their sub-streams of the whole job -- for several) are run one after the other
    and reduced with reduce_job; the result must equal the one-call run of the job in every bit of hist, hist2 and stats."""
    import torch
    from paper_2012_00963_b200 import _shard
    cfg = W.scaled(W.config(idx), 150_001, n_snap=n_snap, n_clouds=n_clouds)
    run, n, world = cfg["run"], cfg["run"]["n_photons"], 3
    clouds = [P.pdv_cloud_create(c) for c in cfg["clouds"]]
    nc, ns, nb = len(clouds), len(cfg["t_snap"]), run["n_bins"]
    total = n * world if scaling == "weak" else n
    whole = P.pdv_mc_run(clouds, cfg["t_snap"], total, 19, run)
    acc_h = torch.zeros((nc * ns, nb), dtype=torch.float64)
    acc_h2 = torch.zeros_like(acc_h)
    parts = []
    for rank in range(world):
        pl = _shard.plan(nc, ns, n, rank, world, scaling)
        r = P.pdv_mc_run([clouds[i] for i in pl["clouds"]], [cfg["t_snap"][j] for j in pl["snaps"]], pl["n_photons"], 19,
                         dict(run, first_photon_id=pl["first_photon_id"], unit_streams=pl["unit_ids"]))
        h, h2, st = _shard.reduce_job(torch.from_numpy(r.hist.reshape(-1, nb)), torch.from_numpy(r.hist2.reshape(-1, nb)),
                                      r.stats.reshape(-1), pl["unit_ids"], nc * ns)
        acc_h += h
        acc_h2 += h2
        parts.append(st)
    st = _shard.merge_stats(parts)
    assert np.array_equal(acc_h.numpy(), whole.hist.reshape(-1, nb)) and np.array_equal(acc_h2.numpy(), whole.hist2.reshape(-1, nb))
    for k in st.dtype.names:
        assert np.array_equal(st[k], whole.stats.reshape(-1)[k]), k


def test_second_production_instantiation_gives_the_same_tallies(P):
    """The ALT instantiations must not change a single bit.  Several classes: a cloud whose class guide is
    clean runs ALT alone, and the plain instantiation when a cloud with a flagged guide cell (config 5's tiny classes) rides in
    the same launch.  One class: a thin cloud runs one draw per pass alone, and four (long histories) next to a thick cloud.
    unit_streams gives the unit the same sub-stream in both launches."""
    for probe, other in ((W.config(2)["clouds"][0], W.config(4)["clouds"][0]),                 # 16 classes: clean / flagged guide
                         (W.config(1)["clouds"][0], W._cloud(20.0, 6.0, 2000.0, diameter_um=1.0))):     # one class: tau 1.9 / 108
        run = dict(W.config(1)["run"], n_bins=512, v_hi=9000.0)
        n = 300_007
        a, b = P.pdv_cloud_create(probe), P.pdv_cloud_create(other)
        poly = len(probe.get("diameters", [])) > 1 or "lognormal" in probe
        alone = P.pdv_mc_run([a], [2.0e-6], n, 77, dict(run, unit_streams=[5]))
        alt_alone = P.pdv_last_launch_info()["alt"]
        both = P.pdv_mc_run([b, a], [2.0e-6], n, 77, dict(run, unit_streams=[9, 5]))
        alt_both = P.pdv_last_launch_info()["alt"]
        assert alt_alone != alt_both, (poly, alt_alone, alt_both)      # the two launches did run different instantiations
        assert alt_alone == poly
        assert np.array_equal(alone.hist[0, 0], both.hist[1, 0]) and np.array_equal(alone.hist2[0, 0], both.hist2[1, 0])
        for k in alone.stats.dtype.names:
            assert alone.stats[0, 0][k] == both.stats[1, 0][k], k
        assert float(alone.stats[0, 0]["detected"]) > 0


def test_one_class_cloud_inside_a_polydisperse_launch(P):
    """A one-class cloud that rides in a polydisperse launch runs through the class pick (guide of zeros, padded thresholds,
    its table and albedo stored twice): its spectrum must agree with the one-class kernel's (another random word map, so
    statistically) and its weights must be conserved exactly."""
    mono, poly = W.config(1)["clouds"][0], W.config(2)["clouds"][0]
    run = W.config(1)["run"]
    n = 2_000_000
    a, b = P.pdv_cloud_create(mono), P.pdv_cloud_create(poly)
    alone = P.pdv_mc_run([a], [3.0e-6], n, 31, run)
    assert not (P.pdv_last_launch_info()["variant"] & 1)
    mixed = P.pdv_mc_run([b, a], [3.0e-6], n, 32, run)
    assert P.pdv_last_launch_info()["variant"] & 1 and P.pdv_last_launch_info()["alt"]
    assert mixed.conservation_residual()[1, 0] == 0.0
    res = compare(alone.hist[0, 0], alone.hist2[0, 0], n, mixed.hist[1, 0], mixed.hist2[1, 0], n)
    assert res["ndf"] >= 50 and res["worst"] < 5.0, res["z"]
    for k in ("detected", "escaped", "absorbed_particles", "absorbed_surface"):
        x, y = float(alone.stats[0, 0][k]) / n, float(mixed.stats[1, 0][k]) / n
        assert abs(x - y) < 5 * math.sqrt((x + y) / n), (k, x, y)
    assert int(mixed.stats[1, 0]["particle_events"]) == pytest.approx(int(alone.stats[0, 0]["particle_events"]), rel=5e-3)


def test_detection_queue_under_full_load(P):
    """Every history is a detection (aperture 2 pi, empty cloud: each photon reflects once and leaves): every lane of a warp pushes
    on the detection queue in the same pass, the queue is tallied every pass, and the counts must still be exact."""
    params = W._cloud(0.0, 4.0, 2000.0, diameter_um=5.0)
    run = dict(W.config(0)["run"], aperture_sr=2.0 * math.pi, n_bins=64)
    n = 1_000_003
    r = P.pdv_mc_run([P.pdv_cloud_create(params)], [2.0e-6], n, 5, run)
    s = r.stats[0, 0]
    assert int(s["histories"]) == n and int(s["surface_reflections"]) == n and int(s["particle_events"]) == 0
    assert r.conservation_residual()[0, 0] == 0.0
    # weight R per history, all inside [0, v_fs): Q31 sums are exact
    assert float(s["detected"]) + float(s["underflow"]) + float(s["overflow"]) == pytest.approx(0.6 * n, rel=1e-6)
    assert r.hist[0, 0].sum() == pytest.approx(float(s["detected"]), rel=1e-12)


def test_photon_count_limit_of_the_fixed_point_tallies(P):
    cfg = W.config(1)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    with pytest.raises(P.PdvError) as e:                       # 2^33 photons of weight 1 in one tally = 2^64: wraps
        P.pdv_mc_run([c], cfg["t_snap"], 2 ** 33, 1, cfg["run"])
    assert e.value.status == 1 and "2^33" in str(e.value)


def test_full_size_config2_in_bench_launch_configuration(P):
    """BASELINE.json configs[1] at full size (1e8 photons, default launch shape = what bench.py times): invariants
    that hold at any size, plus parity against the stored 4e8-history oracle run (tests/golden/oracle_hist_cfg2.json)."""
    cfg = W.config(1)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = cfg["run"]["n_photons"]
    r = P.pdv_mc_run([c], cfg["t_snap"], n, cfg["run"]["seed"], cfg["run"])
    s = r.stats[0, 0]
    assert s["histories"] == n
    # 1e8 * 2^31 exceeds 2^53: the double sum of exact Q31 terms may round in the last bits only
    assert abs(r.conservation_residual()[0, 0]) < 1e-6
    assert r.hist.sum() == pytest.approx(s["detected"], rel=1e-12)
    o = load_golden("cfg2")
    n_o = o.n_photons
    assert n_o >= 4 * n and o.run["n_bins"] == cfg["run"]["n_bins"]
    res = _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, o, min_ndf=300)
    top_g = (s["detected"] + s["underflow"] + s["overflow"] + s["escaped"]) / n
    top_o = (o.stats["detected"] + o.stats["underflow"] + o.stats["overflow"] + o.stats["escaped"]) / n_o
    assert top_g == pytest.approx(top_o, rel=1e-3)                  # integrated backscatter, north_star
    a, b = s["detected"] / n, o.stats["detected"] / n_o
    assert abs(a - b) < 5 * math.sqrt(a / n + b / n_o)
    assert s["particle_events"] / n == pytest.approx(o.stats["particle_events"] / n_o, rel=2e-3)


def test_full_size_configs_3_4_5(P):
    """The other BASELINE.json configs at their full photon counts in the default launch shape: config 3 (16 classes) as a
    slice of 4 of its 200 snapshots at 1e8 photons each, config 4 in full (48 clouds x 1e7), config 5 in full (1e9 photons,
    64-bit photon ids, roulette after 200 events).  Invariants that hold at any size, and parity of sampled outputs against
    the stored oracle runs of 1e8 ... 4e8 histories (tests/golden/oracle_hist_*.json, written by make_oracle_hists.py from
    oracle/ alone): at these sizes the 5 sigma band is the GPU's own noise, and reading R23 holds with 25 effective counts
    for every config."""
    # ---- config 3
    cfg = W.config(2)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = cfg["run"]["n_photons"]
    t4 = cfg["t_snap"][:2] + cfg["t_snap"][-2:]
    r = P.pdv_mc_run([c], t4, n, cfg["run"]["seed"], cfg["run"])
    o = load_golden("cfg3")
    assert o.n_photons >= 4 * n
    for i in range(4):
        s = r.stats[0, i]
        assert s["histories"] == n and abs(r.conservation_residual()[0, i]) < 1e-6
        _assert_hist_parity(r.hist[0, i], r.hist2[0, i], n, o, min_ndf=300)
        _assert_stats_parity(s, n, o)
        assert s["particle_events"] / n == pytest.approx(o.stats["particle_events"] / o.n_photons, rel=1e-3)
    res = compare(r.hist[0, 0], r.hist2[0, 0], n, r.hist[0, 3], r.hist2[0, 3], n)       # t = 0.5 us against t = 10 us (R16)
    assert res["worst"] < 5.0
    # ---- config 4
    cfg = W.config(3)
    clouds = [P.pdv_cloud_create(p) for p in cfg["clouds"]]
    n = cfg["run"]["n_photons"]
    r = P.pdv_mc_run(clouds, cfg["t_snap"], n, cfg["run"]["seed"], cfg["run"])
    # 1e7 * 2^31 exceeds 2^53: the double sum of exact Q31 terms may round in the last bit
    assert np.all(r.stats["histories"] == n) and np.all(np.abs(r.conservation_residual()) < 1e-7)
    assert np.allclose(r.hist.sum(axis=2), r.stats["detected"], rtol=1e-12)
    # ALL 48 clouds against stored oracle runs: four of them (thin ... thick: tau 1.2, 0.9, 9.3, 18.6) at 1e8 oracle histories,
    # the other 44 at 2e7 (20 chunks of 1e6: batch-means variances for the statistics)
    for i in range(48):
        oo = load_golden(f"cfg4_cloud{i:02d}")
        big = i in (3, 22, 36, 44)
        assert oo.n_photons >= (10 if big else 2) * n and oo.tau_ext == pytest.approx(clouds[i].info()["tau_ext"], rel=1e-9)
        _assert_hist_parity(r.hist[i, 0], r.hist2[i, 0], n, oo, min_ndf=50 if big else 20)
        _assert_stats_parity(r.stats[i, 0], n, oo)
        assert r.stats[i, 0]["particle_events"] / n == pytest.approx(oo.stats["particle_events"] / oo.n_photons, rel=3e-3), i
    # ---- config 5
    cfg = W.config(4)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = cfg["run"]["n_photons"]
    assert n == 10 ** 9
    run = dict(cfg["run"], first_photon_id=2 ** 32 - 12345)       # the id range straddles 2^32
    r = P.pdv_mc_run([c], cfg["t_snap"], n, cfg["run"]["seed"], run)
    s = r.stats[0, 0]
    assert s["histories"] == n and abs(r.conservation_residual()[0, 0]) < 1e-5
    assert r.hist.sum() == pytest.approx(s["detected"], rel=1e-12)
    oo = load_golden("cfg5")                                      # 4e8 oracle histories
    _assert_hist_parity(r.hist[0, 0], r.hist2[0, 0], n, oo, min_ndf=300)
    _assert_stats_parity(s, n, oo, same_game=False)
    top_g = (s["detected"] + s["underflow"] + s["overflow"] + s["escaped"]) / n
    top_o = (oo.stats["detected"] + oo.stats["underflow"] + oo.stats["overflow"] + oo.stats["escaped"]) / oo.n_photons
    assert top_g == pytest.approx(top_o, abs=5 * math.sqrt(top_o / oo.n_photons))


@pytest.mark.parametrize("m0,d_um", [(1.0, 5.0), (3.0, 2.0), (2.0, None)])
def test_mean_path_invariance_on_the_device(P, m0, d_um):
    """The CUDA transport against a theorem, with no reference implementation in the loop (pin P16 on the device):
    non-absorbing particles (real index 1.5, full Mie table), lossless Lambertian bottom, diffuse illumination
    (launch_model 1) => per history <particle events> = 4 tau_ext, <surface reflections> = 1, and the light that leaves is
    Lambertian: P(mu_exit >= mu_a) = 1 - mu_a^2.  1e8 histories: the 5 sigma band is 1.5e-4 of the value, far below anything
    a wrong constant, a biased uniform or a sloppy approximation in the fp32 flight could hide in."""
    base = W._cloud(m0, 4.0, 2000.0, diameter_um=d_um) if d_um else W._cloud(m0, 4.0, 2000.0, lognormal=(3.0, 0.5, 16))
    params = dict(base, m_re=1.5, m_im=0.0, surface_model=1, surface_reflectivity=1.0)      # d_um None: 16 size classes
    c = P.pdv_cloud_create(params)
    tau = c.info()["tau_ext"]
    run = dict(W.config(1)["run"], aperture_sr=0.1, v_lo=-20000.0, v_hi=20000.0, launch_model=1)
    _, rec = P.pdv_mc_trace(c, 0, 200_000, 5, run)                      # spread of the per-history counts
    sd_ev, sd_rf = rec["n_scatter"].std(), rec["n_reflect"].std()
    n = 100_000_000
    r = P.pdv_mc_run([c], [1e-6], n, 77, run)
    s = r.stats[0, 0]
    assert s["histories"] == n and s["absorbed_particles"] == 0.0 and s["absorbed_surface"] == 0.0
    assert s["particle_events"] / n == pytest.approx(4.0 * tau, abs=5 * sd_ev / math.sqrt(n))
    assert s["surface_reflections"] / n == pytest.approx(1.0, abs=5 * sd_rf / math.sqrt(n))
    p_in = 1.0 - (1.0 - 0.1 / (2 * math.pi)) ** 2
    assert (s["detected"] + s["underflow"] + s["overflow"]) / n == pytest.approx(p_in, abs=5 * math.sqrt(p_in / n))
    # not vacuous: the collimated beam on the same cloud does not give 4 tau
    r0 = P.pdv_mc_run([c], [1e-6], 1_000_000, 77, dict(run, launch_model=0))
    assert abs(r0.stats[0, 0]["particle_events"] / 1e6 - 4.0 * tau) > 20 * sd_ev / math.sqrt(1e6)       # 2.7 % ... 12 % off


@pytest.mark.parametrize("poly", [False, True])
def test_rigid_cloud_doppler_telescopes_on_the_device(P, poly):
    """Pin P17 on the device, no reference in the loop: particles and free surface all at v = 2000 m/s => the Doppler
    velocity of a history is (1 + mu_exit) v / 2 whatever its length, so all detected weight lies in
    [(1 + mu_a)/2 v, v] = [1984.08, 2000.00] m/s.  fp32 accumulation over up to ~70 events: edges within 0.05 m/s."""
    base = W.config(2 if poly else 1)["clouds"][0]
    params = dict(base, area_mass=2.0e-2, profile_kind=1, prof_v=np.array([2000.0, 2000.002]), prof_cum_mass=np.array([0.0, 1.0]),
                  vmax_ratio=1.000001)
    c = P.pdv_cloud_create(params)
    n, nb, lo, hi = 20_000_000, 2000, 1950.0, 2050.0               # 0.05 m/s per bin (16 classes + 8000 bins exceed shared memory)
    run = dict(W.config(1)["run"], n_bins=nb, v_lo=lo, v_hi=hi)
    r = P.pdv_mc_run([c], [1e-6], n, 17, run)
    s = r.stats[0, 0]
    assert s["particle_events"] / n > 5.0 and s["max_events_in_history"] > 50
    assert s["underflow"] == 0.0 and s["overflow"] == 0.0 and s["detected"] / n > 0.01
    mu_a = 1.0 - 0.1 / (2 * math.pi)
    centres = lo + (np.arange(nb) + 0.5) * (hi - lo) / nb
    inside = (centres > 0.5 * (1 + mu_a) * 2000.0 - 0.05) & (centres < 2000.002 + 0.05)
    h = r.hist[0, 0]
    assert h[~inside].sum() == 0.0 and h[inside].sum() == pytest.approx(s["detected"], rel=1e-12)
    _, rec = P.pdv_mc_trace(c, 0, 300_000, 17, run)
    out = rec["fate"] != 2
    resid = rec["vt"][out].astype(np.float64) - 0.5 * (1.0 + rec["mu_exit"][out].astype(np.float64)) * 2000.0
    assert np.max(np.abs(resid)) < 0.05


def test_double_scattering_closed_form_on_the_device(P):
    """Pin P20 on the device, no reference run in the loop: the histories of exactly two particle events of an isotropic cloud
    with a velocity profile over an absorbing surface, traced on the GPU, against the 4-D Gauss-Legendre quadrature of
    tests/test_oracle_mc.py (count, first three moments of v~, coarse histogram)."""
    from test_oracle_mc import _double_scatter_quadrature
    params = dict(W.config(1)["clouds"][0], phase_model=1, surface_reflectivity=0.0)
    oc = ocloud.build_cloud(params, phase_override=ocloud.isotropic_quantile_table(1024)[None, :])       # tables of the closed form
    om, omega_sr, n = float(oc.omega0[0]), 2.0, 4_000_000
    mu_a = 1.0 - omega_sr / (2.0 * math.pi)
    run = dict(W.config(1)["run"], aperture_sr=omega_sr)
    _, rec = P.pdv_mc_trace(P.pdv_cloud_create(params), 0, n, 2012, run)
    sel = (rec["fate"] == 0) & (rec["n_scatter"] == 2) & (rec["n_reflect"] == 0)
    assert np.allclose(rec["weight"][sel], om ** 2, rtol=1e-6)
    vt, wt = _double_scatter_quadrature(oc, om, mu_a)
    W0 = float(wt.sum())
    p_sel = W0 / om ** 2
    assert sel.sum() == pytest.approx(n * p_sel, abs=5 * math.sqrt(n * p_sel))
    v_g = rec["vt"][sel].astype(np.float64)
    for k in (1, 2, 3):
        m_q = float(np.sum(wt * vt ** k)) / W0
        sig = float(np.std(v_g ** k)) / math.sqrt(sel.sum())
        assert float(np.mean(v_g ** k)) == pytest.approx(m_q, abs=5 * sig + 2e-4 * m_q), k
    edges = np.linspace(0.0, 6000.0, 25)
    h_q, _ = np.histogram(vt, bins=edges, weights=wt)
    h_g, _ = np.histogram(v_g, bins=edges)
    big = h_q * n > 2000 * om ** 2
    assert big.sum() >= 8
    expect = n * h_q[big] / om ** 2
    assert np.all(np.abs(h_g[big] - expect) <= 5 * np.sqrt(expect) + 0.01 * expect)


def test_rare_paths_stress_many_short_runs(P):
    """Short runs that spend most of their time in the rare paths (roulette kill / survive, analog absorption,
    single-scatter truncation, drained-queue lanes) in varying order: every run must complete, conserve weight
    exactly and be bit-reproducible.  (A first version of the kernel faulted intermittently here.)"""
    cfg = W.config(1)
    kws = [dict(max_events=3, roulette_survival=0.5), dict(), dict(mode=1), dict(single_scatter_only=1),
           dict(mode=1, max_events=2, roulette_survival=0.3), dict(max_events=1, roulette_survival=0.1)]
    ref = {}
    for rep in range(6):
        for i in (np.arange(len(kws)) + rep) % len(kws):
            c = P.pdv_cloud_create(cfg["clouds"][0])
            n = 200_000 + 1000 * int(i)
            r = P.pdv_mc_run([c], cfg["t_snap"], n, 77, dict(cfg["run"], **kws[i]))
            assert r.stats[0, 0]["histories"] == n and r.conservation_residual()[0, 0] == 0.0
            key = int(i)
            if key in ref:
                assert np.array_equal(ref[key], r.hist)
            ref[key] = r.hist
