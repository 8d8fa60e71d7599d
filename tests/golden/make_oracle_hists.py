#!/usr/bin/env python
"""Writes the stored oracle histograms tests/golden/oracle_hist_*.json -- calls ONLY oracle/ (and pdv_workloads for the inputs).

    python tests/golden/make_oracle_hists.py [name ...]        # default: all; takes ~35 min on 8 cores

The full-size GPU parity tests (tests/test_gpu_parity.py::test_full_size_*) compare 1e8 ... 1e9-history GPU runs with the oracle.
An oracle run the test can afford live (a few 1e6 histories) leaves the comparison without power where it matters (the tolerance
5 sqrt(var_gpu + var_cpu) is then the oracle's own noise), so the oracle is run ONCE here at >= 1e8 histories per spectrum and its
tallies are stored as text: hist = sum of weights per bin, hist2 = sum of squared weights per bin, the run statistics, the photon
count, the generator (rng_mode 0 = xoshiro256**, unrelated to the GPU's Philox) and the seed.  Nothing here is computed by, or read
from, the CUDA path.  One spectrum per cloud is enough: in vacuum the expected spectrum does not depend on the snapshot time
(reading R16), so the same stored spectrum serves every snapshot of config 3.
"""
from __future__ import annotations

import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import pdv_workloads as W  # noqa: E402
from oracle import cloud as ocloud  # noqa: E402
from oracle import mc as omc  # noqa: E402

SEED = 20201203
CHUNK = 50_000_000          # histories per oracle call (ids [k CHUNK, (k+1) CHUNK)): bounds the size of one call

# name -> (BASELINE.json config index, cloud index, histories)
JOBS = {
    "cfg2": (1, 0, 400_000_000),
    "cfg3": (2, 0, 400_000_000),
    "cfg4_cloud03": (3, 3, 100_000_000),
    "cfg4_cloud22": (3, 22, 100_000_000),
    "cfg4_cloud36": (3, 36, 100_000_000),
    "cfg4_cloud44": (3, 44, 100_000_000),
    "cfg5": (4, 0, 400_000_000),
    # the other 44 clouds of config 4 at 2e7 histories each (twice the GPU's 1e7), in chunks of 1e6: filled in below
    # row f4 (pdv_workloads.gas_spectrogram, bench.py --config 6): with a gas the spectrum depends on the snapshot time (DESIGN.md
    # R38), so a spectrum is stored per snapshot: the first and the last of the 20.  ("gas", snapshot index, histories)
    "f4gas_snap00": ("gas", 0, 100_000_000),
    "f4gas_snap19": ("gas", 19, 100_000_000),
    # the same last snapshot with 1024 depth bins instead of the workload's 256 (the product limit for 16 classes in a gas, pdv.h):
    # oracle against oracle, the two stored runs bound the discretisation error of the 256 bins at 1e8 histories
    # (tests/test_oracle_gas.py).  ("gas", snapshot index, histories, depth bins)
    "f4gas_snap19_nd1024": ("gas", 19, 100_000_000, 1024),
}
for _i in range(48):
    if f"cfg4_cloud{_i:02d}" not in JOBS:
        JOBS[f"cfg4_cloud{_i:02d}"] = (3, _i, 20_000_000)
SMALL_CHUNK = 1_000_000     # chunk of the 2e7-history jobs: 20 chunks for the batch-means variances


def make(name: str) -> str:
    idx, ci, n = JOBS[name][:3]
    n_depth = JOBS[name][3] if len(JOBS[name]) > 3 else None
    chunk = CHUNK if n >= 100_000_000 else SMALL_CHUNK
    gas = None
    if idx == "gas":
        from oracle import gas as ogas
        cfg, snap, ci = W.gas_spectrogram(), ci, 0
        par = cfg["clouds"][0]
        oc = ocloud.build_cloud(par)
        gas = ogas.build_tables(oc, par, cfg["t_snap"][snap], n_depth or par["n_depth_bins"])
    else:
        cfg = W.config(idx)
        oc = ocloud.build_cloud(cfg["clouds"][ci])
    run = dict(cfg["run"], seed=SEED)
    hist = hist2 = None
    stats: dict = {}
    t0 = time.time()
    chunk_stats = []        # statistics of every chunk: batch-means variances of the weights that are far from 0/1 per history
    for first in range(0, n, chunk):
        r = omc.run(oc, run, n_photons=min(chunk, n - first), first_id=first, gas=gas)
        hist = r.hist if hist is None else hist + r.hist
        hist2 = r.hist2 if hist2 is None else hist2 + r.hist2
        chunk_stats.append({k: (int(v) if isinstance(v, int) else float(v)) for k, v in r.stats.items()})
        for k, v in r.stats.items():
            stats[k] = max(stats.get(k, 0), v) if k == "max_events_in_history" else stats.get(k, 0) + v
    out = {
        "what": "oracle/ (fp64 CPU Monte-Carlo) tallies; written by tests/golden/make_oracle_hists.py; no value comes from the CUDA path",
        "workload": cfg["name"], "config_index": idx, "cloud_index": ci, "t_snap": (gas["t"] if gas else None), "n_photons": n, "seed": SEED, "rng_mode": 0,
        "run": {k: run[k] for k in ("n_bins", "v_lo", "v_hi", "aperture_sr", "mode", "max_events", "roulette_survival")},
        "n_depth_bins": (n_depth or cfg["clouds"][0].get("n_depth_bins")), "tau_ext": oc.tau_ext, "seconds": round(time.time() - t0, 1), "threads": os.cpu_count(),
        "stats": {k: (int(v) if isinstance(v, int) else float(v)) for k, v in stats.items()},
        "chunk": chunk, "chunk_stats": chunk_stats,
        "hist": [float(x) for x in hist], "hist2": [float(x) for x in hist2],
    }
    path = os.path.join(HERE, f"oracle_hist_{name}.json")
    with open(path, "w") as f:
        json.dump(out, f, separators=(",", ":"))
        f.write("\n")
    return path


if __name__ == "__main__":
    for nm in (sys.argv[1:] or list(JOBS)):
        t = time.time()
        p = make(nm)
        print(f"{nm}: {p} ({time.time() - t:.0f} s)", flush=True)
