"""Multi-GPU plumbing of the photon path: histories are independent and keyed by photon id, so
a run shards by id range with NO data-path collective; the only exchange is one sum of the additive tallies
(histograms, sums of squared weights, counters) at the end of a run.  One process per GPU; `torch.distributed`
(NCCL on GPUs, gloo in the CPU tests) carries that sum.  No method arithmetic lives here.
"""
from __future__ import annotations

import numpy as np


def shard_photons(n_total: int, rank: int, world: int, first_photon_id: int = 0) -> tuple[int, int]:
    """Contiguous id range of `rank`: (first id, count).  The ranges of all ranks tile
    [first_photon_id, first_photon_id + n_total) exactly; the first n_total % world ranks get one more."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n_total >= 0")
    base, rem = divmod(int(n_total), world)
    count = base + (1 if rank < rem else 0)
    start = int(first_photon_id) + rank * base + min(rank, rem)
    return start, count


def shard_units(n_units: int, rank: int, world: int) -> range:
    """Whole (cloud, snapshot) units per rank (configs 3 and 4): unit u goes to rank u % world."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n_units >= 0")
    return range(rank, n_units, world)


def plan(n_clouds: int, n_snap: int, n_photons: int, rank: int, world: int, scaling: str = "weak",
         first_photon_id: int = 0) -> dict:
    """What `rank` of `world` processes runs of a job of n_clouds x n_snap units with n_photons histories per unit
    (SURVEY.md 8(e)).  Returns {"clouds": cloud indices, "snaps": snapshot indices, "unit_ids": index of each local unit in the
    whole job (row-major over the local clouds x snaps grid; pass it as run["unit_streams"]), "first_photon_id", "n_photons"}.

    weak    every rank runs ALL units with n_photons histories on its own id range [first + rank n, first + (rank+1) n):
            the job grows with the number of GPUs (n_photons * world histories per unit in total).
    strong  the job is fixed.  One unit (configs 2, 5): the id range is split (shard_photons).  Several units (configs 3, 4):
            whole units per rank, unit u to rank u % world (shard_units) -- along the snapshots when the job has one cloud,
            along the clouds when it has one snapshot; a clouds x snapshots grid is split along the clouds.
    In every case the union of what the ranks run is a job whose tallies are the bit-exact sum / concatenation of theirs."""
    if scaling not in ("weak", "strong"):
        raise ValueError("scaling must be 'weak' or 'strong'")
    all_c, all_s = list(range(n_clouds)), list(range(n_snap))
    if scaling == "weak":
        c, s_, first, n = all_c, all_s, int(first_photon_id) + rank * int(n_photons), int(n_photons)
    elif n_clouds * n_snap == 1:
        c, s_ = all_c, all_s
        first, n = shard_photons(n_photons, rank, world, first_photon_id)
    elif n_clouds == 1:
        c, s_, first, n = all_c, list(shard_units(n_snap, rank, world)), int(first_photon_id), int(n_photons)
    else:
        c, s_, first, n = list(shard_units(n_clouds, rank, world)), all_s, int(first_photon_id), int(n_photons)
    return {"clouds": c, "snaps": s_, "unit_ids": [i * n_snap + j for i in c for j in s_], "first_photon_id": first, "n_photons": n}


ADDITIVE_STATS = ("detected", "underflow", "overflow", "escaped", "absorbed_particles", "absorbed_surface",
                  "roulette_killed", "roulette_gained", "truncated", "histories", "particle_events",
                  "surface_reflections")


def allreduce_tallies(hist, hist2=None, group=None):
    """In-place sum over ranks of the additive tallies (torch tensors, CPU for gloo / CUDA for NCCL).
    Tallies are integer multiples of 2^-31 below 2^53 * 2^-31, so the float64 sums are exact and the result
    does not depend on the reduction order (bit-identical to a one-GPU run over the union of the id ranges)."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return
    dist.all_reduce(hist, op=dist.ReduceOp.SUM, group=group)
    if hist2 is not None:
        dist.all_reduce(hist2, op=dist.ReduceOp.SUM, group=group)


def merge_stats(stats_list):
    """Merges per-rank structured stats arrays (STATS_DTYPE) of the same units: additive fields are summed,
    max_events_in_history is the maximum."""
    out = np.array(stats_list[0], copy=True)
    for s in stats_list[1:]:
        for k in ADDITIVE_STATS:
            out[k] = out[k] + s[k]
        out["max_events_in_history"] = np.maximum(out["max_events_in_history"], s["max_events_in_history"])
    return out


def reduce_job(hist, hist2, stats, unit_ids, n_units: int, group=None):
    """All ranks end up with the tallies of the WHOLE job: `hist`, `hist2` are this rank's [n_local, n_bins] float64 torch
    tensors (CPU for gloo, CUDA for NCCL), `stats` its structured numpy array [n_local] (STATS_DTYPE), `unit_ids` the index of
    each local unit in the job.  Rows are scattered into zero [n_units, n_bins] tensors and summed over ranks (ranks that ran
    the same unit on different id ranges add up, ranks that ran different units fill different rows); the statistics are
    reduced the same way, additive fields summed, max_events_in_history by maximum.  All sums are exact: tallies are integer
    multiples of 2^-31 below 2^22, counters are integers below 2^53.  Returns (hist, hist2, stats) of the job."""
    import torch
    import torch.distributed as dist
    idx = torch.as_tensor(list(unit_ids), dtype=torch.long, device=hist.device)
    nb = hist.shape[-1]
    out = torch.zeros((2, n_units, nb), dtype=torch.float64, device=hist.device)
    out[0].index_add_(0, idx, hist.reshape(-1, nb))
    out[1].index_add_(0, idx, hist2.reshape(-1, nb))
    st = np.asarray(stats).reshape(-1)
    add = torch.zeros((n_units, len(ADDITIVE_STATS)), dtype=torch.float64, device=hist.device)
    mx = torch.zeros(n_units, dtype=torch.float64, device=hist.device)
    if len(st):
        add.index_add_(0, idx, torch.as_tensor(np.stack([st[k].astype(np.float64) for k in ADDITIVE_STATS], axis=1), device=hist.device))
        mx.index_copy_(0, idx, torch.as_tensor(st["max_events_in_history"].astype(np.float64), device=hist.device))
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(add, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(mx, op=dist.ReduceOp.MAX, group=group)
    job = np.zeros(n_units, dtype=st.dtype)
    a, m = add.cpu().numpy(), mx.cpu().numpy()
    for i, k in enumerate(ADDITIVE_STATS):
        job[k] = a[:, i]
    job["max_events_in_history"] = m
    return out[0], out[1], job
