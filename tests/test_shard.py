"""Host logic of the multi-GPU path: photon-id / unit sharding and the one
all-reduce of the additive tallies, on 2 gloo ranks on the CPU.  No method arithmetic is involved: each rank's
"tallies" are a deterministic integer function of the photon ids it owns, so the reduced result must equal the
single-rank result bit for bit for any split."""
import os
import socket

import numpy as np
import pytest

from paper_2012_00963_b200._shard import ADDITIVE_STATS, allreduce_tallies, merge_stats, shard_photons, shard_units


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
