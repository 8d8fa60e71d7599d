"""GPU parity for SURVEY.md 8(f) row f4, ejecta in a gas environment (readings R35-R38, which are NOT the paper's:
PAPER.md:409 names the case as future work without an equation).  The CUDA path (transport_kernel<..., DM = 3>, one device
image per (cloud, snapshot) unit) against the fp64 oracle (oracle/gas.py + the gas branch of pdv_oracle_mc.c), snapshot by
snapshot, with the north_star tolerance; reading R16 (time invariance) must now FAIL with gas and still hold without."""
import math

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud as ocloud
from oracle import gas as ogas
from oracle import mc as omc

from histcmp import compare

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("_library_is_built")]


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2012_00963_b200 as P
    return P


def _parity(g_hist, g_hist2, n_g, o, min_ndf):
    res = compare(g_hist, g_hist2, n_g, o.hist, o.hist2, o.n_photons)
    assert res["ndf"] >= min_ndf and res["worst"] < 5.0, (res["ndf"], res["worst"])
    assert res["chi2"] < res["ndf"] + 6 * math.sqrt(2 * res["ndf"]) + 10
    return res


@pytest.mark.parametrize("idx,rho_g,n_depth,kw", [(1, 8.0, 1024, dict()), (1, 8.0, 1024, dict(mode=1)), (2, 5.0, 256, dict()),
                                                  (4, 3.0, 256, dict())])
def test_gas_units_match_the_oracle_snapshot_by_snapshot(P, idx, rho_g, n_depth, kw):
    """One size (config 2's cloud), 16 sizes (config 3's), and the thick roulette case (config 5's cloud), each at three snapshot
    times in ONE launch: every spectrum against the oracle's run of the same unit."""
    cfg = W.config(idx)
    params = dict(cfg["clouds"][0], gas_density=rho_g, drag_coefficient=0.5, n_depth_bins=n_depth)
    run = dict(cfg["run"], **kw)
    times = [0.7e-6, 3e-6, 9e-6]
    c = P.pdv_cloud_create(params)
    n = 1_500_000 if idx != 4 else 500_000
    r = P.pdv_mc_run([c], times, n, 61, run)
    oc = ocloud.build_cloud(params)
    peaks = []
    for j, t in enumerate(times):
        o = omc.run(oc, dict(run, seed=1234 + j), n_photons=n, gas=ogas.build_tables(oc, params, t, n_depth))
        _parity(r.hist[0, j], r.hist2[0, j], n, o, min_ndf=30)
        s = r.stats[0, j]
        assert s["histories"] == n and r.conservation_residual()[0, j] == 0.0
        for key in ("detected", "escaped", "absorbed_particles", "absorbed_surface"):
            a, b = float(s[key]) / n, o.stats[key] / n
            assert abs(a - b) < 5 * math.sqrt((max(a, 1e-12) + max(b, 1e-12)) / n), (key, a, b)
        if "max_events" not in run or not run["max_events"]:
            assert s["particle_events"] / n == pytest.approx(o.stats["particle_events"] / n, rel=0.02)
        peaks.append(int(np.argmax(np.convolve(r.hist[0, j], np.ones(9) / 9, mode="same"))))
    # R38: the spectrum changes with time -- first and last snapshot differ far beyond the noise
    res = compare(r.hist[0, 0], r.hist2[0, 0], n, r.hist[0, 2], r.hist2[0, 2], n)
    assert res["worst"] > 15.0


def test_vacuum_limit_and_time_invariance(P):
    """gas_density -> 0 through the gas kernel: the same spectrum as the vacuum kernel (statistically: other code path, same
    physics), whatever the snapshot time (R16 holds again); gas_density = 0 IS the vacuum path: bit-identical."""
    cfg = W.config(2)
    base = dict(cfg["clouds"][0], n_depth_bins=256)
    run, n, times = cfg["run"], 1_500_000, [1e-6, 8e-6]
    v = P.pdv_mc_run([P.pdv_cloud_create(base)], times, n, 5, run)
    z = P.pdv_mc_run([P.pdv_cloud_create(dict(base, gas_density=0.0, drag_coefficient=0.5))], times, n, 5, run)
    assert np.array_equal(v.hist, z.hist) and np.array_equal(v.hist2, z.hist2)
    for k in v.stats.dtype.names:
        assert np.array_equal(v.stats[k], z.stats[k]), k
    g = P.pdv_mc_run([P.pdv_cloud_create(dict(base, gas_density=1e-9, drag_coefficient=0.5))], times, n, 6, run)
    for (ha, h2a), (hb, h2b) in (((g.hist[0, 0], g.hist2[0, 0]), (v.hist[0, 0], v.hist2[0, 0])),
                                 ((g.hist[0, 1], g.hist2[0, 1]), (v.hist[0, 1], v.hist2[0, 1])),
                                 ((g.hist[0, 0], g.hist2[0, 0]), (g.hist[0, 1], g.hist2[0, 1]))):
        res = compare(ha, h2a, n, hb, h2b, n)
        assert res["worst"] < 5.0 and res["chi2"] < res["ndf"] + 6 * math.sqrt(2 * res["ndf"]) + 10
    assert g.stats[0, 0]["particle_events"] / n == pytest.approx(v.stats[0, 0]["particle_events"] / n, rel=5e-3)


def test_gas_and_vacuum_clouds_share_a_launch_and_runs_are_reproducible(P):
    """A launch with a gas cloud runs every unit through the gas kernel (vacuum clouds with L = infinity); results do not depend
    on the launch shape or on how the id range is split."""
    cfg = W.config(1)
    pg = dict(cfg["clouds"][0], gas_density=8.0, drag_coefficient=0.5)
    pv = dict(cfg["clouds"][0])
    run, n, times = cfg["run"], 400_001, [2e-6, 5e-6]
    clouds = [P.pdv_cloud_create(pg), P.pdv_cloud_create(pv)]
    a = P.pdv_mc_run(clouds, times, n, 9, run)
    b = P.pdv_mc_run(clouds, times, n, 9, dict(run, blocks_per_sm=1, threads_per_block=128))
    assert np.array_equal(a.hist, b.hist) and np.array_equal(a.stats["particle_events"], b.stats["particle_events"])
    h1 = P.pdv_mc_run(clouds, times, 150_000, 9, run)
    h2 = P.pdv_mc_run(clouds, times, n - 150_000, 9, dict(run, first_photon_id=150_000))
    assert np.array_equal(a.hist, h1.hist + h2.hist)
    assert np.all(a.conservation_residual() == 0.0)
    # the vacuum cloud inside the gas launch: statistically the vacuum kernel's spectrum, at both times
    v = P.pdv_mc_run([clouds[1]], times, n, 10, run)
    for j in range(2):
        assert compare(a.hist[1, j], a.hist2[1, j], n, v.hist[0, j], v.hist2[0, j], n)["worst"] < 5.0
    # and the gas cloud's spectrum has moved towards v_fs: far less detected weight above 1.5 v_fs than in vacuum
    high = lambda h: float(h[256:].sum() / h.sum())
    assert high(a.hist[0, 1]) < 0.6 * high(a.hist[1, 1])


def test_gas_requests_the_kernel_does_not_implement_are_refused(P):
    cfg = W.config(1)
    c = P.pdv_cloud_create(dict(cfg["clouds"][0], gas_density=8.0, drag_coefficient=0.5))
    for bad in (dict(single_scatter_only=1), dict(launch_model=1)):
        with pytest.raises(P.PdvError):
            P.pdv_mc_run([c], [1e-6], 1000, 1, dict(cfg["run"], **bad))
    with pytest.raises(P.PdvError):
        P.pdv_mc_trace(c, 0, 1000, 1, cfg["run"])
    with pytest.raises(P.PdvError):
        P.pdv_cloud_create(dict(cfg["clouds"][0], gas_density=8.0, drag_coefficient=0.0))
    with pytest.raises(P.PdvError):
        P.pdv_cloud_create(dict(cfg["clouds"][0], gas_density=8.0, drag_coefficient=0.5, depth_model=1))


def test_full_size_gas_spectrogram_against_stored_oracle_runs(P):
    """Row f4 at the size and in the launch bench.py --config 6 times (20 snapshots x 1e7 photons of the 16-class cloud in a gas, one
    launch, every snapshot a unit with its own image): the first and the last spectrum against the stored 1e8-history oracle runs of
    those two units (tests/golden/oracle_hist_f4gas_snap*.json, written by make_oracle_hists.py from oracle/ alone)."""
    from histcmp import load_golden
    cfg = W.gas_spectrogram()
    run, n = cfg["run"], cfg["run"]["n_photons"]
    r = P.pdv_mc_run([P.pdv_cloud_create(cfg["clouds"][0])], cfg["t_snap"], n, run["seed"], run)
    assert (P.pdv_last_launch_info()["variant"] >> 8) == 3 and P.pdv_last_launch_info()["variant"] & 1
    assert np.all(r.conservation_residual() == 0.0)
    for j, name in ((0, "f4gas_snap00"), (len(cfg["t_snap"]) - 1, "f4gas_snap19")):
        o = load_golden(name)
        res = _parity(r.hist[0, j], r.hist2[0, j], n, o, min_ndf=100)
        s = r.stats[0, j]
        for key in ("detected", "escaped", "absorbed_particles", "absorbed_surface"):
            a, b = float(s[key]) / n, o.stats[key] / o.n_photons
            assert abs(a - b) < 5 * math.sqrt(max(a, 1e-12) / n + max(b, 1e-12) / o.n_photons), (key, a, b)
        assert s["particle_events"] / n == pytest.approx(o.stats["particle_events"] / o.n_photons, rel=2e-3)
        assert abs((float(s["detected"]) + float(s["underflow"]) + float(s["overflow"]) + float(s["escaped"])) / n
                   - (o.stats["detected"] + o.stats["underflow"] + o.stats["overflow"] + o.stats["escaped"]) / o.n_photons) \
            < 1e-3 * (o.stats["detected"] + o.stats["escaped"]) / o.n_photons + 5 * math.sqrt(0.5 / n)
    # the two spectra are far apart (R38): the stored runs themselves differ by many sigma
    a, b = load_golden("f4gas_snap00"), load_golden("f4gas_snap19")
    assert compare(a.hist, a.hist2, a.n_photons, b.hist, b.hist2, b.n_photons)["worst"] > 50
