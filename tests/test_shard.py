"""Host logic of the multi-GPU path: photon-id / unit sharding and the one
all-reduce of the additive tallies, on 2 gloo ranks on the CPU.  No method arithmetic is involved: each rank's
"tallies" are a deterministic integer function of the photon ids it owns, so the reduced result must equal the
single-rank result bit for bit for any split."""
import os
import socket

import numpy as np
import pytest

from paper_2012_00963_b200._shard import ADDITIVE_STATS, allreduce_tallies, merge_stats, plan, reduce_job, shard_photons, shard_units


def test_shard_photons_tiles_the_id_range_exactly():
    for n_total in (0, 1, 7, 100, 10**9 + 7):
        for world in (1, 2, 3, 8):
            at = 5
            for rank in range(world):
                first, count = shard_photons(n_total, rank, world, first_photon_id=5)
                assert first == at and count in (n_total // world, n_total // world + 1)
                at += count
            assert at == 5 + n_total
    with pytest.raises(ValueError):
        shard_photons(10, 2, 2)


def test_shard_units_partitions_all_units():
    for n_units in (0, 1, 48, 200):
        for world in (1, 2, 8):
            seen = sorted(u for r in range(world) for u in shard_units(n_units, r, world))
            assert seen == list(range(n_units))


def _fake_tallies(first, count, n_bins):
    """Integer tallies in units of 2^-31 as float64 (what finalize_kernel writes): bin = id % n_bins, weight = a Q31
    integer derived from the id."""
    ids = np.arange(first, first + count, dtype=np.uint64)
    w = ((ids * np.uint64(2654435761)) % np.uint64(2**31)).astype(np.float64) / 2.0**31
    hist = np.bincount((ids % np.uint64(n_bins)).astype(np.int64), weights=w, minlength=n_bins)
    hist2 = np.bincount((ids % np.uint64(n_bins)).astype(np.int64), weights=np.floor(w * w * 2.0**31) / 2.0**31, minlength=n_bins)
    return hist, hist2


def _worker(rank, world, port, n_total, n_bins, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    first, count = shard_photons(n_total, rank, world)
    h, h2 = _fake_tallies(first, count, n_bins)
    th, th2 = torch.from_numpy(h.copy()), torch.from_numpy(h2.copy())
    allreduce_tallies(th, th2)
    np.save(os.path.join(out_dir, f"h_{rank}.npy"), th.numpy())
    np.save(os.path.join(out_dir, f"h2_{rank}.npy"), th2.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_allreduce_of_sharded_tallies_equals_single_rank_bit_for_bit(tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    n_total, n_bins, world = 200_001, 64, 2
    mp.spawn(_worker, args=(world, port, n_total, n_bins, str(tmp_path)), nprocs=world, join=True)
    ref_h, ref_h2 = _fake_tallies(0, n_total, n_bins)
    for rank in range(world):
        assert np.array_equal(np.load(tmp_path / f"h_{rank}.npy"), ref_h)
        assert np.array_equal(np.load(tmp_path / f"h2_{rank}.npy"), ref_h2)


def test_merge_stats_sums_additive_fields_and_takes_the_max():
    from paper_2012_00963_b200 import STATS_DTYPE
    a = np.zeros(3, dtype=STATS_DTYPE)
    b = np.zeros(3, dtype=STATS_DTYPE)
    for i, k in enumerate(ADDITIVE_STATS):
        a[k] = i + 1
        b[k] = 10 * (i + 1)
    a["max_events_in_history"] = [5, 9, 2]
    b["max_events_in_history"] = [7, 3, 2]
    m = merge_stats([a, b])
    for i, k in enumerate(ADDITIVE_STATS):
        assert np.all(m[k] == 11 * (i + 1))
    assert list(m["max_events_in_history"]) == [7, 9, 2]


# ---------------------------------------------------------------------------------------------------------------------------
# The sharding arithmetic bench.py runs (plan + reduce_job), on 2 gloo ranks.  The "tallies" of a unit are a deterministic
# integer function of (unit id, photon id), as the library's are of (unit sub-stream, photon id): whatever the split, the
# reduced job must equal the one-rank job bit for bit.
def _fake_unit(unit, first, count, n_bins):
    ids = np.arange(first, first + count, dtype=np.uint64)
    key = ids * np.uint64(2654435761) + np.uint64(unit) * np.uint64(40503)
    w = (key % np.uint64(2**31)).astype(np.float64) / 2.0**31
    b = (key % np.uint64(n_bins)).astype(np.int64)
    hist = np.bincount(b, weights=w, minlength=n_bins)
    hist2 = np.bincount(b, weights=np.floor(w * w * 2.0**31) / 2.0**31, minlength=n_bins)
    return hist, hist2, int((key % np.uint64(7)).sum()), int((key % np.uint64(97)).max()) if count else 0


def _fake_job(n_clouds, n_snap, n_photons, n_bins, rank, world, scaling):
    from paper_2012_00963_b200 import STATS_DTYPE
    pl = plan(n_clouds, n_snap, n_photons, rank, world, scaling)
    n_loc = len(pl["unit_ids"])
    h, h2, st = np.zeros((n_loc, n_bins)), np.zeros((n_loc, n_bins)), np.zeros(n_loc, dtype=STATS_DTYPE)
    for k, u in enumerate(pl["unit_ids"]):
        h[k], h2[k], ev, mx = _fake_unit(u, pl["first_photon_id"], pl["n_photons"], n_bins)
        st[k]["histories"], st[k]["particle_events"], st[k]["max_events_in_history"] = pl["n_photons"], ev, mx
        st[k]["detected"] = h[k].sum()
    return pl, h, h2, st


def _job_worker(rank, world, port, cases, n_bins, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    for ci, (nc, ns, n, scaling) in enumerate(cases):
        pl, h, h2, st = _fake_job(nc, ns, n, n_bins, rank, world, scaling)
        jh, jh2, jst = reduce_job(torch.from_numpy(h), torch.from_numpy(h2), st, pl["unit_ids"], nc * ns)
        np.save(os.path.join(out_dir, f"job{ci}_h_{rank}.npy"), jh.numpy())
        np.save(os.path.join(out_dir, f"job{ci}_h2_{rank}.npy"), jh2.numpy())
        np.save(os.path.join(out_dir, f"job{ci}_st_{rank}.npy"), jst)
    dist.barrier()
    dist.destroy_process_group()


CASES = [(1, 1, 100_003, "strong"),      # one unit: the id range is split (configs 2, 5)
         (1, 7, 20_000, "strong"),       # one cloud, several snapshots: whole snapshots per rank (config 3)
         (5, 1, 20_000, "strong"),       # several clouds, one snapshot: whole clouds per rank (config 4, the sweeps)
         (3, 2, 10_000, "strong"),       # a grid: split along the clouds
         (2, 3, 15_001, "weak")]         # every rank runs every unit on its own id range


def test_plan_covers_the_job_exactly():
    for nc, ns, n, scaling in CASES:
        for world in (1, 2, 3, 8):
            units, photons = {}, 0
            for rank in range(world):
                pl = plan(nc, ns, n, rank, world, scaling)
                assert pl["unit_ids"] == [i * ns + j for i in pl["clouds"] for j in pl["snaps"]]
                for u in pl["unit_ids"]:
                    units.setdefault(u, []).append((pl["first_photon_id"], pl["n_photons"]))
            assert sorted(units) == list(range(nc * ns))
            for u, ranges in units.items():
                ranges.sort()
                at = 0
                for first, count in ranges:                  # the id ranges of a unit tile [0, total) without gap or overlap
                    assert first == at
                    at += count
                assert at == (n * world if scaling == "weak" else n)
    with pytest.raises(ValueError):
        plan(1, 1, 10, 0, 1, "both")


def test_reduced_job_of_two_ranks_equals_the_one_rank_job_bit_for_bit(tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    n_bins, world = 48, 2
    mp.spawn(_job_worker, args=(world, port, CASES, n_bins, str(tmp_path)), nprocs=world, join=True)
    for ci, (nc, ns, n, scaling) in enumerate(CASES):
        total = n * world if scaling == "weak" else n
        _, h, h2, st = _fake_job(nc, ns, total, n_bins, 0, 1, "strong")          # the whole job on one rank
        for rank in range(world):
            assert np.array_equal(np.load(tmp_path / f"job{ci}_h_{rank}.npy"), h), (ci, rank)
            assert np.array_equal(np.load(tmp_path / f"job{ci}_h2_{rank}.npy"), h2), (ci, rank)
            jst = np.load(tmp_path / f"job{ci}_st_{rank}.npy")
            for k in ("histories", "particle_events", "max_events_in_history", "detected"):
                assert np.array_equal(jst[k], st[k]), (ci, rank, k)


# ---------------------------------------------------------------------------------------- cost-balanced strong split
def _check_balanced_tiling(costs, nc, ns, n, world):
    from paper_2012_00963_b200._shard import plan_balanced
    seen = {}
    cost_of_rank = []
    for rank in range(world):
        segs = plan_balanced(costs, nc, ns, n, rank, world, first_photon_id=1000)
        c = 0.0
        for sg in segs:
            assert sg["unit_ids"] == [i * ns + j for i in sg["clouds"] for j in sg["snaps"]] and sg["n_photons"] > 0
            for u in sg["unit_ids"]:
                seen.setdefault(u, []).append((sg["first_photon_id"], sg["n_photons"]))
                c += costs[u] * sg["n_photons"]
        assert len({u for sg in segs for u in sg["unit_ids"]}) == sum(len(sg["unit_ids"]) for sg in segs)     # a unit once per rank
        cost_of_rank.append(c)
    assert sorted(seen) == list(range(nc * ns))
    for u, ranges in seen.items():                           # the id ranges of every unit tile [1000, 1000 + n) exactly
        ranges.sort()
        at = 1000
        for first, count in ranges:
            assert first == at
            at += count
        assert at == 1000 + n
    return cost_of_rank


def test_balanced_plan_tiles_the_job_exactly_for_any_costs():
    rng = np.random.default_rng(5)
    for nc, ns in ((1, 7), (5, 1), (3, 4), (48, 1), (1, 200), (2, 1)):
        for world in (1, 2, 3, 8):
            for n in (1, 17, 100_003):
                costs = list(rng.uniform(0.5, 120.0, size=nc * ns))
                cost_of_rank = _check_balanced_tiling(costs, nc, ns, n, world)
                if n >= 100_003:                             # long units: the cuts fall where the cost line says
                    assert max(cost_of_rank) <= 1.001 * (sum(cost_of_rank) / world)
    _check_balanced_tiling([0.0, 0.0, 3.0], 3, 1, 10, 2)     # units of no cost go along
    from paper_2012_00963_b200._shard import plan_balanced
    with pytest.raises(ValueError):
        plan_balanced([1.0], 2, 1, 10, 0, 1)


@pytest.mark.usefixtures("_library_is_built")
def test_balanced_plan_of_config4_and_the_fig13_sweep_at_8_gpus():
    """with unit u -> rank u % world, config 4 at 8 GPUs gave ranks 0-1 every 1 um cloud and ranks 6-7
    every 10 um cloud: max / mean estimated cost 2.3.  Cut along the library's own cost line it is 1 by construction (<= 1.1
    asked); the estimate comes from the library (pdv_estimated_flights, no GPU needed), not from a copy of its formula."""
    import paper_2012_00963_b200 as P
    import pdv_workloads as W
    for cfg in (W.config(3), W.paper_sweep("fig13_15", n_photons=10 ** 7)):
        clouds = [P.pdv_cloud_create(c) for c in cfg["clouds"]]
        costs = [c.estimated_flights(cfg["run"]) for c in clouds]
        assert min(costs) > 1.0 and max(costs) / min(costs) > 1.5               # heterogeneous, else the test says nothing
        n = cfg["run"]["n_photons"]
        by_rank = _check_balanced_tiling(costs, len(clouds), 1, n, 8)
        assert max(by_rank) / (sum(by_rank) / 8) <= 1.001
        modulo = [sum(costs[u] * n for u in range(r, len(costs), 8)) for r in range(8)]
        assert max(modulo) / (sum(modulo) / 8) > (2.0 if len(costs) == 48 else 1.1)      # what the old split did: 2.3 and 1.14
    # the estimate follows the run options it depends on
    c = clouds[0]
    assert c.estimated_flights(dict(max_events=5, roulette_survival=0.1)) < c.estimated_flights({})
    assert c.estimated_flights(dict(single_scatter_only=1)) <= 3.0


def _device_reduce_worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    from paper_2012_00963_b200 import STATS_DTYPE
    from paper_2012_00963_b200._shard import plan_balanced
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nc, ns, n, nb = 5, 1, 20_001, 16
    costs = [3.0, 40.0, 7.5, 90.0, 12.0]
    segs = plan_balanced(costs, nc, ns, n, rank, world)
    rows_h, rows_h2, rows_st, ids = [], [], [], []
    for sg in segs:
        for u in sg["unit_ids"]:
            h, h2, ev, mx = _fake_unit(u, sg["first_photon_id"], sg["n_photons"], nb)
            st = np.zeros(1, dtype=STATS_DTYPE)
            st["histories"], st["particle_events"], st["max_events_in_history"], st["detected"] = sg["n_photons"], ev, mx, h.sum()
            rows_h.append(h); rows_h2.append(h2); rows_st.append(st); ids.append(u)
    h = torch.from_numpy(np.array(rows_h).reshape(-1, nb))
    h2 = torch.from_numpy(np.array(rows_h2).reshape(-1, nb))
    st = np.concatenate(rows_st) if rows_st else np.zeros(0, dtype=STATS_DTYPE)
    st_u8 = torch.from_numpy(np.frombuffer(st.tobytes(), dtype=np.uint8).copy())
    jh, jh2, jst = reduce_job(h, h2, st_u8, ids, nc * ns)                 # statistics as the raw records: the device path
    kh, kh2, kst = reduce_job(h, h2, st, ids, nc * ns)                    # and as a numpy array: the host path
    jst = jst.numpy().view(STATS_DTYPE)
    assert np.array_equal(jh.numpy(), kh.numpy()) and np.array_equal(jh2.numpy(), kh2.numpy())
    for k in STATS_DTYPE.names:
        assert np.array_equal(jst[k], kst[k]), k
    np.save(os.path.join(out_dir, f"bal_h_{rank}.npy"), jh.numpy())
    np.save(os.path.join(out_dir, f"bal_st_{rank}.npy"), jst)
    dist.barrier()
    dist.destroy_process_group()


def test_balanced_job_of_two_ranks_reduces_to_the_one_rank_job_bit_for_bit(tmp_path):
    """gloo, world 2: units split by photon id at the rank boundary, reduced with the statistics kept as raw records (what
    bench.py does on the device); every rank ends with the tallies of the one-rank job."""
    import torch.multiprocessing as mp
    from paper_2012_00963_b200 import STATS_DTYPE
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_device_reduce_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    nc, n, nb = 5, 20_001, 16
    want_h = np.array([_fake_unit(u, 0, n, nb)[0] for u in range(nc)])
    for rank in range(2):
        assert np.array_equal(np.load(tmp_path / f"bal_h_{rank}.npy"), want_h)
        st = np.load(tmp_path / f"bal_st_{rank}.npy")
        assert np.array_equal(st["histories"], np.full(nc, n, dtype=np.uint64))
        assert np.array_equal(st["particle_events"], np.array([_fake_unit(u, 0, n, nb)[2] for u in range(nc)], dtype=np.uint64))
        assert np.array_equal(st["max_events_in_history"], np.array([_fake_unit(u, 0, n, nb)[3] for u in range(nc)], dtype=np.uint64))
