"""GPU: the launches bench.py times, checked row by row, and the links between the traced kernel, the production
instantiations and the generator's published vectors ("Next round" item 1).

  * pin P13: raw blocks of the device Philox4x32-10 through each of its three key paths against the
    published known-answer vectors (tests/golden/philox4x32_10_kat.txt);
  * pdv_mc_trace (TRACE instantiation, compared history by history with the oracle in test_gpu_parity.py) and pdv_mc_run (the
    production instantiations BENCH times) give the SAME integer tallies for the same seed, unit stream and id range: the
    history-by-history evidence carries over to the kernels that are timed;
  * config 3 as BENCH launches it -- ALL 200 snapshots in one launch, more units than blocks (the stacked
    spectrogram is the paper's product): every row against the stored 4e8-history oracle spectrum, rows mutually consistent.
"""
import math
import os

import numpy as np
import pytest

import pdv_workloads as W

from histcmp import compare, load_golden

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


def test_device_philox_known_answers_through_every_key_path(P):
    """Pin P13: the generator the kernels run, not a copy of it -- philox4x32_10<uint4*>, <SharedKeys>, <ParamKeys> are the
    functions transport_kernel calls (csrc/pdv_kernels.cu), here applied to the published counters and keys."""
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        seed = w[4] | (w[5] << 32)
        # the vector's counter, plus neighbours so that several threads and a ragged tail run
        ctr = np.array([w[0:4]] + [[k, 0, 7, k * k] for k in range(1, 200)], dtype=np.uint32)
        outs = P.pdv_philox_blocks(ctr, seed)
        for o, name in zip(outs, ("static shared keys", "shared address", "kernel parameters")):
            assert [int(x) for x in o[0]] == w[6:10], (name, [hex(int(x)) for x in o[0]])
        assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
        assert len({tuple(r) for r in outs[0].tolist()}) == 200          # distinct counters, distinct blocks
        n += 1
    assert n == 3
    a, b, c = P.pdv_philox_blocks(np.zeros((0, 4), dtype=np.uint32), 1)
    assert a.shape == (0, 4)


def _mono(m0, d_um, beta=4.0):
    return W._cloud(m0, beta, 2000.0, diameter_um=d_um)


# (cloud, run overrides, expected bits of pdv_last_launch_info()["variant"] & 0x33 = poly | analog | roulette | ALT, name)
CASES = [
    (W.config(1)["clouds"][0], dict(), 0, "one class, short histories: <0,0,0,0,0,0,0> (config 2, the headline)"),
    (_mono(10.0, 2.0), dict(), 32, "one class, long histories: <0,...,ALT> (config 4's thick clouds)"),
    (W.config(2)["clouds"][0], dict(), 1 | 32, "16 classes, clean class guide: <1,...,ALT> (config 3, Figs. 13-15 sweep)"),
    (W.config(4)["clouds"][0], dict(), 1, "16 classes, flagged class guide, no roulette: <1,0,0,0,0,0,0>"),
    (W.config(4)["clouds"][0], dict(max_events=200, roulette_survival=0.1), 1 | 16, "16 classes + roulette: <1,...,ROUL> (config 5)"),
    (W.config(1)["clouds"][0], dict(mode=1), 2, "one class, analog absorption: <0,1,...>"),
]


@pytest.mark.parametrize("case", range(len(CASES)))
def test_trace_kernel_and_production_kernels_tally_the_same_bits(P, case):
    params, kw, want_variant, name = CASES[case]
    run = dict(W.config(1)["run"], n_bins=512, v_hi=3.0 * params["v_fs"], **kw)
    c = P.pdv_cloud_create(params)
    n, seed, unit, first = 120_011, 97531, 5, 1_000_003
    run_t = dict(run, first_photon_id=first)
    rt, rec = P.pdv_mc_trace(c, unit, n, seed, run_t)
    assert P.pdv_last_launch_info()["variant"] & 8, "pdv_mc_trace did not run the TRACE instantiation"
    rp = P.pdv_mc_run([c], [2.0e-6], n, seed, dict(run_t, unit_streams=[unit]))
    v = P.pdv_last_launch_info()["variant"]
    assert v & 8 == 0 and (v & 0x33) == want_variant and (v >> 8) == 0, (name, hex(v))
    assert np.array_equal(rt.hist, rp.hist) and np.array_equal(rt.hist2, rp.hist2), name
    for k in rt.stats.dtype.names:
        assert np.array_equal(rt.stats[k], rp.stats[k]), (name, k)
    assert int(rp.stats[0, 0]["histories"]) == n and rp.hist.sum() > 0
    # and the records add up to the tallies they came with
    det = rec["fate"] == 0
    assert abs(float(rec["weight"][det].astype(np.float64).sum()) - rt.hist.sum()) < 1e-3 * rt.hist.sum() + 1e-3


def _stats_sigma(a, b, n_a, n_b):
    return math.sqrt(max(a, 1e-12) / n_a + max(b, 1e-12) / n_b)


def test_config3_all_200_snapshots_in_one_launch(P):
    """bench.py --config 2's launch shape: 200 (cloud, snapshot) units on 148 blocks -- units shorter than a block's share of the
    cost line, the wrap-around walk, block_start.  1e6 photons per snapshot (the GPU's noise is then 20x the golden's)."""
    cfg = W.config(2)
    c = P.pdv_cloud_create(cfg["clouds"][0])
    n = 1_000_000
    assert len(cfg["t_snap"]) == 200
    r = P.pdv_mc_run([c], cfg["t_snap"], n, cfg["run"]["seed"], cfg["run"])
    info = P.pdv_last_launch_info()
    assert info["grid"] < 200, "the point of this test is more units than blocks"
    assert (info["variant"] & 0x33) == (1 | 32)                     # the instantiation BENCH times for config 3
    o = load_golden("cfg3")
    assert np.all(r.stats["histories"] == n)
    assert np.all(r.conservation_residual() == 0.0)                 # 1e6 * 2^31 < 2^53: exact in double
    assert np.allclose(r.hist.sum(axis=2), r.stats["detected"], rtol=1e-12)
    # 200 rows x ~100 merged bins = 2e4 comparisons of Poisson-like counts.  Merged bins of 25 effective counts (reading R23, what
    # the one-spectrum tests use) are too skewed for that many: a count of 25 exceeds 5 sigma upwards with probability ~1e-5, not
    # 3e-7, and one row in the first run of this test had a bin at 5.9 sigma.  So: bins of >= 100 effective counts, the 5 sigma
    # bar applied to the family (no bin of the 2e4 beyond 6 sigma, at most 12 beyond 4 -- a Gaussian family expects 1.3), chi-square
    # per row, and the strict north_star bar (25 counts, 5 sigma per bin) on the SUM of the rows below.
    worst, chi2, ndf, beyond4 = 0.0, 0.0, 0, 0
    for i in range(200):
        res = compare(r.hist[0, i], r.hist2[0, i], n, o.hist, o.hist2, o.n_photons, min_eff=100.0)
        assert res["ndf"] >= 60 and res["worst"] < 6.0, (i, res["ndf"], res["worst"])
        assert res["chi2"] < res["ndf"] + 6 * math.sqrt(2 * res["ndf"]) + 10, (i, res["chi2"], res["ndf"])
        worst, chi2, ndf = max(worst, res["worst"]), chi2 + res["chi2"], ndf + res["ndf"]
        beyond4 += int(np.sum(np.abs(res["z"]) > 4.0))
        s = r.stats[0, i]
        for key in ("detected", "escaped", "absorbed_particles", "absorbed_surface"):
            a, b = float(s[key]) / n, o.stats[key] / o.n_photons
            assert abs(a - b) < 5 * _stats_sigma(a, b, n, o.n_photons), (i, key, a, b)
        assert s["particle_events"] / n == pytest.approx(o.stats["particle_events"] / o.n_photons, rel=0.01)
    assert beyond4 <= 12, beyond4
    # the 200 rows together: chi2 over ~200 x ndf degrees of freedom stays within 5 sigma of its mean
    assert abs(chi2 - ndf) < 5 * math.sqrt(2 * ndf), (chi2, ndf)
    # all rows are draws of ONE spectrum (time invariance in vacuum, R16 / pin P10) from independent streams:
    assert len({r.hist[0, i].tobytes() for i in range(200)}) == 200
    for i, j in ((0, 199), (1, 100), (57, 143), (148, 149), (147, 148)):            # incl. the rows around the block count
        res = compare(r.hist[0, i], r.hist2[0, i], n, r.hist[0, j], r.hist2[0, j], n, min_eff=100.0)
        assert res["worst"] < 5.0, (i, j, res["worst"])
    # the sum of the rows is a 2e8-history spectrum: the sharpest comparison with the 4e8-history oracle run
    res = compare(r.hist[0].sum(axis=0), r.hist2[0].sum(axis=0), 200 * n, o.hist, o.hist2, o.n_photons)
    assert res["ndf"] >= 300 and res["worst"] < 5.0 and res["chi2"] < res["ndf"] + 6 * math.sqrt(2 * res["ndf"]) + 10
    # bit-identical to the same units run one launch each (the unit's sub-stream is its index in the job)
    for i in (0, 148, 199):
        one = P.pdv_mc_run([c], [cfg["t_snap"][i]], n, cfg["run"]["seed"], dict(cfg["run"], unit_streams=[i]))
        assert np.array_equal(one.hist[0, 0], r.hist[0, i]) and one.stats[0, 0] == r.stats[0, i]


def test_cloud_creation_does_not_wait_for_a_run_on_another_stream(P):
    """pdv_cloud_create used to synchronise the whole device whenever it recycled the buffer of a destroyed cloud, and uploaded
    with a blocking copy: creating a cloud waited for every stream's work.  Now it waits for the runs that read the OLD cloud
    only (an event) and uploads on a stream of its own.  Here: a 1e9-history run (config 5, ~0.25 s) is enqueued on stream A;
    while it runs, config 4's 48 clouds are created and destroyed on the host -- from recycled buffers -- in a few milliseconds,
    and A's run is still in flight afterwards.  A's tallies equal those of an undisturbed run, bit for bit."""
    import time
    import torch
    torch.cuda.set_device(0)
    cfg5, cfg4 = W.config(4), W.config(3)
    c5 = P.pdv_cloud_create(cfg5["clouds"][0])
    run5, nb = cfg5["run"], cfg5["run"]["n_bins"]
    # round 0: the 48 buffers exist, have been read by a run (their events are recorded) and are back in the cache
    first = [P.pdv_cloud_create(p) for p in cfg4["clouds"]]
    P.pdv_mc_run(first, cfg4["t_snap"], 1000, 1, cfg4["run"])
    for c in first:
        c.destroy()
    ref = P.pdv_mc_run([c5], cfg5["t_snap"], 10 ** 9, 5, run5)
    a = torch.cuda.Stream()
    h, h2 = (torch.zeros((1, 1, nb), dtype=torch.float64, device="cuda") for _ in range(2))
    st = torch.zeros(P.STATS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    done = torch.cuda.Event()
    P.pdv_mc_run_device([c5], cfg5["t_snap"], 10 ** 9, 5, run5, h, h2, st, stream=a.cuda_stream)
    done.record(a)
    t0 = time.perf_counter()
    for _ in range(2):
        again = [P.pdv_cloud_create(p) for p in cfg4["clouds"]]
        for c in again:
            c.destroy()
    dt = time.perf_counter() - t0
    still_running = not done.query()
    torch.cuda.synchronize()
    assert still_running, f"the 1e9-history run had finished after {dt * 1e3:.1f} ms of cloud creation: nothing was tested"
    assert dt < 0.1, f"creating and destroying 2 x 48 clouds took {dt * 1e3:.1f} ms while a run was in flight on another stream"
    assert np.array_equal(h.cpu().numpy(), ref.hist) and np.array_equal(h2.cpu().numpy(), ref.hist2)
    assert st.cpu().numpy().view(P.STATS_DTYPE)[0] == ref.stats[0, 0]


def test_launch_info_is_kept_per_stream(P):
    import torch
    torch.cuda.set_device(0)
    mono, poly = W.config(1), W.scaled(W.config(2), 300_000, n_snap=2)
    cm, cp = P.pdv_cloud_create(mono["clouds"][0]), P.pdv_cloud_create(poly["clouds"][0])
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ha, ha2 = (torch.zeros((1, 1, 512), dtype=torch.float64, device="cuda") for _ in range(2))
    hb, hb2 = (torch.zeros((1, 2, 512), dtype=torch.float64, device="cuda") for _ in range(2))
    P.pdv_mc_run_device([cm], mono["t_snap"], 3_000_000, 1, mono["run"], ha, ha2, None, stream=sa.cuda_stream)
    P.pdv_mc_run_device([cp], poly["t_snap"], 300_000, 1, poly["run"], hb, hb2, None, stream=sb.cuda_stream)
    ia, ib = P.pdv_last_launch_info(stream=sa.cuda_stream), P.pdv_last_launch_info(stream=sb.cuda_stream)
    last = P.pdv_last_launch_info()
    torch.cuda.synchronize()
    assert ia["variant"] & 1 == 0 and ib["variant"] & 1 == 1              # one class on A, sixteen on B
    assert ia["transport_ms"] > 0 and ib["transport_ms"] > 0 and ia["n_kernels"] == 2 and ib["n_kernels"] == 2
    assert last["variant"] == ib["variant"] and last["transport_ms"] == ib["transport_ms"]
    other = torch.cuda.Stream()
    assert P.pdv_last_launch_info(stream=other.cuda_stream)["n_kernels"] == 0


def test_phase_table_error_at_spectrum_level_and_fig6_cases(P):
    """Row f2 at the level of the SPECTRUM.  The headline rests on one approximation, the inverse-CDF
    phase table D_1024 in place of the paper's rejection sampling on the exact Mie function; pdv_phase_sampling_check bounds its
    error on cos(theta), this test bounds its consequence.  Config 2 at its full 1e8 histories is run with D_1024 (the default),
    D_4096 and D_256 in one launch: the interpolation error of the table falls 16x with each step (it is quadratic in the cell
    width), so if D_1024 moved the spectrum, D_256 against D_4096 would show 16x that.  All three spectra agree bin by bin within
    the 5 sigma of their own noise at 1e8 histories (100x the statistics of the CPU pin P12), and so do the integrated rates.
    Then the paper's Fig. 6: Case 1 (Mie) against Case 2 (isotropic scattering, same extinction and albedo) at one optical
    thickness in one launch -- the phase function DOES move the spectrum (the comparison above would be blind otherwise); no
    assumption on the direction of the change is made, only that the two differ by far more than the noise."""
    cfg = W.config(1)
    base = cfg["clouds"][0]
    clouds = [P.pdv_cloud_create(dict(base, n_phase_bins=k)) for k in (1024, 4096, 256)]
    n = cfg["run"]["n_photons"]
    r = P.pdv_mc_run(clouds, cfg["t_snap"], n, 31, cfg["run"])
    worst = {}
    for (i, j) in ((0, 1), (2, 1), (0, 2)):
        res = compare(r.hist[i, 0], r.hist2[i, 0], n, r.hist[j, 0], r.hist2[j, 0], n)
        assert res["ndf"] >= 300 and res["worst"] < 5.0, (i, j, res["worst"])
        assert res["chi2"] < res["ndf"] + 6 * math.sqrt(2 * res["ndf"]) + 10, (i, j, res["chi2"], res["ndf"])
        worst[(i, j)] = res["worst"]
        for key in ("detected", "escaped", "absorbed_particles"):
            a, b = float(r.stats[i, 0][key]) / n, float(r.stats[j, 0][key]) / n
            assert abs(a - b) < 5 * _stats_sigma(a, b, n, n), (i, j, key, a, b)
        assert r.stats[i, 0]["particle_events"] / n == pytest.approx(r.stats[j, 0]["particle_events"] / n, rel=1e-3)
    # Fig. 6, Case 1 against Case 2: the same cloud with the Mie phase function and with isotropic scattering
    n6 = 10 ** 7
    mie, iso = P.pdv_cloud_create(base), P.pdv_cloud_create(dict(base, phase_model=1))
    assert mie.info()["tau_ext"] == iso.info()["tau_ext"] and mie.info()["mean_albedo"] == iso.info()["mean_albedo"]
    r6 = P.pdv_mc_run([mie, iso], cfg["t_snap"], n6, 32, cfg["run"])
    res = compare(r6.hist[0, 0], r6.hist2[0, 0], n6, r6.hist[1, 0], r6.hist2[1, 0], n6)
    assert res["worst"] > 20.0 and res["chi2"] > 10 * res["ndf"], (res["worst"], res["chi2"], res["ndf"])


@pytest.mark.parametrize("idx,n_snap,n_clouds", [(3, None, 7), (2, 5, None)])
def test_cost_balanced_shares_of_a_job_reduce_to_the_one_call_job_bit_for_bit(P, idx, n_snap, n_clouds):
    """Row f3 with the round-3 split (_shard.plan_balanced, what `bench.py --gpus N --scaling strong` runs for multi-unit jobs): the
    job is cut into 3 stretches of equal estimated cost (the library's pdv_estimated_flights), units that straddle a rank boundary
    split by photon id.  The three shares are run one after the other on this GPU, each segment one pdv_mc_run call with its units'
    sub-streams of the whole job, and reduced with reduce_job on the raw statistics records (the device path): hist, hist2 and
    every field of stats equal the one-call run of the job."""
    import torch
    from paper_2012_00963_b200 import _shard
    cfg = W.scaled(W.config(idx), 150_001, n_snap=n_snap, n_clouds=n_clouds)
    run, n, world = cfg["run"], cfg["run"]["n_photons"], 3
    clouds = [P.pdv_cloud_create(c) for c in cfg["clouds"]]
    nc, ns, nb = len(clouds), len(cfg["t_snap"]), run["n_bins"]
    whole = P.pdv_mc_run(clouds, cfg["t_snap"], n, 23, run)
    costs = [c.estimated_flights(run) for c in clouds for _ in cfg["t_snap"]]
    acc_h = torch.zeros((nc * ns, nb), dtype=torch.float64)
    acc_h2 = torch.zeros_like(acc_h)
    acc_st = None
    n_split_units = 0
    for rank in range(world):
        segs = _shard.plan_balanced(costs, nc, ns, n, rank, world)
        assert 1 <= len(segs) <= 3 or ns > 1                  # a partial unit at each end and the whole units between them
        rh, rh2, rs, ids = [], [], [], []
        for sg in segs:
            r = P.pdv_mc_run([clouds[i] for i in sg["clouds"]], [cfg["t_snap"][j] for j in sg["snaps"]], sg["n_photons"], 23,
                             dict(run, first_photon_id=sg["first_photon_id"], unit_streams=sg["unit_ids"]))
            rh.append(r.hist.reshape(-1, nb)); rh2.append(r.hist2.reshape(-1, nb)); rs.append(r.stats.reshape(-1)); ids += sg["unit_ids"]
            n_split_units += sum(1 for _ in sg["unit_ids"]) if sg["n_photons"] < n else 0
        st_u8 = torch.from_numpy(np.frombuffer(np.concatenate(rs).tobytes(), dtype=np.uint8).copy())
        h, h2, st = _shard.reduce_job(torch.from_numpy(np.concatenate(rh)), torch.from_numpy(np.concatenate(rh2)), st_u8, ids, nc * ns)
        acc_h += h
        acc_h2 += h2
        st = st.numpy().view(P.STATS_DTYPE)
        acc_st = st if acc_st is None else _shard.merge_stats([acc_st, st])
    assert n_split_units >= 2                                 # units were indeed cut by photon id
    assert np.array_equal(acc_h.numpy(), whole.hist.reshape(-1, nb)) and np.array_equal(acc_h2.numpy(), whole.hist2.reshape(-1, nb))
    for k in acc_st.dtype.names:
        assert np.array_equal(acc_st[k], whole.stats.reshape(-1)[k]), k
