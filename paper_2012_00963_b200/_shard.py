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


def balanced_boundaries(costs, n_photons: int, world: int) -> list[int]:
    """Cuts the job into `world` stretches of equal estimated cost.  The histories of the job are laid on a line, unit after unit
    (row-major), history k of unit u at index u * n_photons + k, each as long as its unit's cost per history (`costs[u]`, e.g.
    Cloud.estimated_flights).  Returns world + 1 non-decreasing indices g_0 = 0 ... g_world = n_units * n_photons; rank r runs
    [g_r, g_r+1).  Pure integer results from the same floats on every rank: every rank computes the same cuts."""
    n_units, n = len(costs), int(n_photons)
    if world < 1 or n < 0 or any(not (c >= 0.0) for c in costs):
        raise ValueError("need world >= 1, n_photons >= 0, costs >= 0")
    w = [float(c) * n for c in costs]
    total = sum(w)
    cuts = [0]
    u, cum = 0, 0.0
    for r in range(1, world):
        x = total * r / world
        while u < n_units and cum + w[u] <= x:
            cum += w[u]
            u += 1
        if u >= n_units or total == 0.0:
            g = n_units * n if total > 0.0 else (n_units * n * r) // world
        else:
            k = int(round((x - cum) / costs[u])) if costs[u] > 0.0 else 0
            g = u * n + min(max(k, 0), n)
        cuts.append(max(g, cuts[-1]))
    cuts.append(n_units * n)
    return cuts


def plan_balanced(costs, n_clouds: int, n_snap: int, n_photons: int, rank: int, world: int, first_photon_id: int = 0) -> list[dict]:
    """Strong scaling by estimated cost: what `rank` runs of a job of n_clouds x n_snap units is a
    contiguous stretch of the cost line of balanced_boundaries; a unit that straddles a rank boundary is split by photon id
    (tallies are additive in id ranges, so the reduced job is bit-identical to the one-process run).  Returns a list of
    SEGMENTS, each one pdv_mc_run call: {"clouds", "snaps", "unit_ids", "first_photon_id", "n_photons"} as in plan().  At most
    one partial unit at each end; the whole units in between are merged into as few calls as their grid shape allows (a run of
    consecutive clouds when the job has one snapshot per cloud, a run of consecutive snapshots of one cloud otherwise)."""
    if len(costs) != n_clouds * n_snap or not (0 <= rank < world):
        raise ValueError("need one cost per unit and 0 <= rank < world")
    n = int(n_photons)
    cuts = balanced_boundaries(costs, n, world)
    g0, g1 = cuts[rank], cuts[rank + 1]
    pieces = []                                               # (unit, first id offset, count)
    if n > 0:
        for u in range(g0 // n, min((g1 + n - 1) // n, n_clouds * n_snap)):
            a, b = max(g0, u * n) - u * n, min(g1, (u + 1) * n) - u * n
            if b > a:
                pieces.append((u, a, b - a))
    segs: list[dict] = []
    for u, a, cnt in pieces:
        i, j = divmod(u, n_snap)
        last = segs[-1] if segs else None
        same_range = last is not None and last["first_photon_id"] == first_photon_id + a and last["n_photons"] == cnt
        if same_range and n_snap == 1 and last["clouds"][-1] == i - 1:
            last["clouds"].append(i)
            last["unit_ids"].append(u)
        elif same_range and last["clouds"] == [i] and last["snaps"][-1] == j - 1:
            last["snaps"].append(j)
            last["unit_ids"].append(u)
        else:
            segs.append({"clouds": [i], "snaps": [j], "unit_ids": [u], "first_photon_id": int(first_photon_id) + a, "n_photons": cnt})
    return segs


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
    if torch.is_tensor(stats):
        return _reduce_job_device(hist, hist2, stats, unit_ids, n_units, group)
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


N_STAT_FLOATS, N_STAT_WORDS = 9, 13      # pdv_run_stats: 9 doubles (weights) + 4 u64 (histories, events, reflections, max events)


def _reduce_job_device(hist, hist2, stats_u8, unit_ids, n_units: int, group=None):
    """reduce_job with the statistics left where pdv_mc_run wrote them: `stats_u8` is the uint8 tensor [n_local * 104] of
    pdv_run_stats records on the tallies' device.  Nothing is copied to the host and nothing synchronises: inside a timed
    multi-GPU step the reduction is three collectives on device tensors.  Returns (hist, hist2, stats) of the job, stats again a
    uint8 tensor of n_units records (`.cpu().numpy().view(STATS_DTYPE)` reads it).  Exact: weights are multiples of 2^-31 summed
    in float64 below 2^53 * 2^-31, counters are summed as int64."""
    import torch
    import torch.distributed as dist
    idx = torch.as_tensor(list(unit_ids), dtype=torch.long, device=hist.device)
    nb = hist.shape[-1]
    n_local = len(idx)
    out = torch.zeros((2, n_units, nb), dtype=torch.float64, device=hist.device)
    out[0].index_add_(0, idx, hist.reshape(-1, nb)[:n_local])
    out[1].index_add_(0, idx, hist2.reshape(-1, nb)[:n_local])
    words = stats_u8[:n_local * 8 * N_STAT_WORDS].view(torch.int64).reshape(n_local, N_STAT_WORDS)
    wf = torch.zeros((n_units, N_STAT_FLOATS), dtype=torch.float64, device=hist.device)
    wi = torch.zeros((n_units, 3), dtype=torch.int64, device=hist.device)
    mx = torch.zeros(n_units, dtype=torch.int64, device=hist.device)
    if n_local:
        wf.index_add_(0, idx, words[:, :N_STAT_FLOATS].view(torch.float64))
        wi.index_add_(0, idx, words[:, N_STAT_FLOATS:N_STAT_FLOATS + 3])
        mx.index_copy_(0, idx, words[:, N_STAT_WORDS - 1].contiguous())      # a unit appears once per rank: a copy is the maximum
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(wf, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(wi, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(mx, op=dist.ReduceOp.MAX, group=group)
    job = torch.cat([wf.view(torch.int64), wi, mx[:, None]], dim=1).contiguous().view(torch.uint8).reshape(-1)
    return out[0], out[1], job
