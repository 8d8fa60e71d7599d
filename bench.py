#!/usr/bin/env python
"""bench.py -- throughput of the Monte-Carlo PDV hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--scaling weak|strong] [--impl b200|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path over one batch of synthetic input: one pdv_mc_run of
BASELINE.json configs[I] (default I = 1: 2 mg/cm^2 tin cloud, 1e8 photons, 512 bins, t = 3 us) followed by pdv_spectrogram
(and pdv_spectrum_peaks for the sweep workload).  Every step uses a new seed.  Rank 0 prints ONE JSON line.

  value      scattering events/s (particle interactions, BASELINE.json "metric"), whole job, cloud tables resident in HBM and
             outputs left in HBM, timed with CUDA events on the launching stream (max over ranks)
  e2e        the same metric through the host-buffer C-ABI calls a user makes: pdv_cloud_create (host tables + H2D; the
             per-class Mie tables come from the library's process-wide memo, which is WARM after the first step) +
             pdv_mc_run into host arrays (D2H inside) + pdv_spectrogram on host arrays, wall clock, with the time of each
             phase (e2e.phases).  e2e.cold is the same with the memo defeated (the wavelength moved by 1e-12 per step, so every
             Mie table is computed again): what a user pays for a cloud of sizes the process has not seen yet
  roofline   transport kernel against the instruction-issue peak (bound "alu": no HBM traffic, no contraction).  frac =
             EXECUTED thread-instructions of one launch (ncu capture under profiles/, keyed by the sha256 of the kernel
             sources) / the launch duration measured here / the issue peak; null when no capture matches the sources.
             frac_model is the hand count of algorithmic instructions per flight (it charges a whole Philox block to every
             flight while the kernel draws one per two or three flights: it exceeds the executed count, context only)
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on this box's host cores, bounded sample of the same workload
  configs    (N = 1, default run) the other BASELINE.json configs and the row-f1 sweep at full size, 2 timed steps each, each
             with ms_per_step, events/s, roofline, cpu_baseline and clocks -- every config is measured by whoever runs this file

    python bench.py --ingest-ncu <csv> --config I [--command "<the ncu command>"] >> profiles/r3_transport_counters.txt
turns the ncu export of ONE transport-kernel launch into the record `roofline` is computed from (no GPU needed).

--impl reference times the oracle itself (there is no reference code).
N > 1 (paper_2012_00963_b200/_shard.py::plan): --scaling weak (default): rank r runs the same number of histories per unit on
photon ids [r n, (r+1) n); --scaling strong: the job is fixed, one-unit configs split the id range, multi-unit configs give
stretches of equal estimated cost to ranks (_shard.plan_balanced: units that straddle a rank boundary are split by photon id).
Either way the only exchange is one reduction of the tallies per step, on device tensors.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import pdv_workloads as W  # noqa: E402

_E2E_COLD_CALLS = [0]            # cold end-to-end legs so far in this process (each uses wavelengths no earlier one used)
METRIC = "scattering events/s"
UNIT = "events/s"

# Algorithmic thread-instructions of ONE flight (one Philox block + free flight + interaction / reflection / exit) on the
# common path, counted from the method's operations, not from what the compiler emitted (DESIGN.md "Roofline",
# table "algorithmic instructions per flight").  A particle event, a surface reflection and the final exit flight are
# one flight each.
ALG_INST_PER_FLIGHT = {"scatter": 96, "reflect": 70, "exit": 64}
COUNTERS_FILES = [os.path.join(ROOT, "profiles", f) for f in ("r3_transport_counters.txt", "r2_transport_counters.txt")]

# ncu metric -> key of a counters record.  The first five are required; the rest describe where the issue slots go
# (north_star: pipe utilisation, warp execution efficiency, shared-memory / atomic throughput) and may be absent from old records.
NCU_METRICS = {
    "smsp__thread_inst_executed.sum": "thread_inst_executed", "smsp__inst_executed.sum": "inst_executed",
    "dram__bytes_read.sum": "dram_bytes_read", "dram__bytes_write.sum": "dram_bytes_write", "gpu__time_duration.sum": "gpu_time_ms",
    "smsp__issue_active.avg.pct_of_peak_sustained_active": "issue_active_pct",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active": "pipe_alu_pct",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed": "pipe_fmaheavy_pct",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active": "pipe_xu_pct",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed": "smem_wavefronts_pct",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum": "smem_wavefronts",
    "sm__warps_active.avg.pct_of_peak_sustained_active": "warps_active_pct",
    "smsp__inst_executed_op_shared_atom.sum": "shared_atom_inst",
}
NCU_REQUIRED = ("thread_inst_executed", "inst_executed", "dram_bytes_read", "dram_bytes_write", "gpu_time_ms")
NCU_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1e-6, "us": 1e-3, "usecond": 1e-3, "ms": 1.0, "msecond": 1.0,
             "nsecond": 1e-6, "second": 1e3, "s": 1e3}


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


# ---------------------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU with NVML every 5 ms while the timed regions run."""

    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int, uuid: str | None = None):
        self.max_mhz = None
        self.reset()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            try:
                self._h = pynvml.nvmlDeviceGetHandleByUUID(uuid if uuid.startswith("GPU-") else "GPU-" + uuid)
            except Exception:
                self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def reset(self):
        self.samples, self.reason_bits, self.power = [], 0, []
        self._stop = threading.Event()

    def _loop(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                self.reason_bits |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(0.005)

    def __enter__(self):
        self._stop.clear()
        if self._nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
            self._thr = None

    def summary(self) -> dict:
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(n for b, n in self.REASONS.items() if self.reason_bits & b),
                "samples": len(self.samples), "power_w_max": max(self.power) if self.power else None}


def _workload(index: int) -> dict:
    """BASELINE.json configs 0..4, 5: the paper's Figs. 13-15 parameter sweep (row f1), 6: ejecta in a gas environment (row f4)."""
    if index == 6:
        return W.gas_spectrogram()
    return W.paper_sweep("fig13_15", n_photons=10 ** 7) if index == 5 else W.config(index)


# ------------------------------------------------------------------------------------------------------ CPU oracle
def _oracle_gas(cfg: dict, oc):
    """Tables of unit 0 of a gas workload (row f4) for the oracle, or None in vacuum."""
    par = cfg["clouds"][0]
    if not par.get("gas_density", 0.0) > 0.0:
        return None
    from oracle import gas as ogas
    return ogas.build_tables(oc, par, cfg["t_snap"][0], par.get("n_depth_bins", 1024))


def oracle_timed(cfg: dict, seconds: float, seed: int):
    """Times the oracle, as it stands, on all host cores for about `seconds` of work on unit 0 of `cfg`."""
    from oracle import cloud as ocloud
    from oracle import mc as omc
    omc.build()
    oc = ocloud.build_cloud(cfg["clouds"][0])
    cores = os.cpu_count() or 1
    run = dict(cfg["run"], seed=seed)
    n0 = 200_000
    gas = _oracle_gas(cfg, oc)
    t = time.perf_counter()
    omc.run(oc, run, n_photons=n0, n_threads=cores, gas=gas)
    dt = max(time.perf_counter() - t, 1e-3)
    n = int(min(max(n0, seconds * n0 / dt), cfg["run"]["n_photons"]))
    t = time.perf_counter()
    r = omc.run(oc, run, n_photons=n, n_threads=cores, first_id=n0, gas=gas)
    dt = time.perf_counter() - t
    return dict(n=n, seconds=dt, events=int(r.stats["particle_events"]), cores=cores)


def _cpu_baseline(cfg: dict, seconds: float, seed: int) -> dict:
    o = oracle_timed(cfg, seconds, seed)
    return {"value": o["events"] / o["seconds"], "unit": UNIT, "cores": o["cores"], "kind": "oracle",
            "histories_per_s": o["n"] / o["seconds"],
            "sample": f"unit 0 of {cfg['name']}: {o['n']} histories in {o['seconds']:.1f} s"}


def run_reference(args):
    """`--impl reference`: the oracle timed on the host cores, each step a bounded sample of the workload."""
    rank = _env_int("RANK", 0)
    if rank != 0:
        return
    from oracle import cloud as ocloud
    from oracle import mc as omc
    omc.build()
    cfg = _workload(args.config)
    oc = ocloud.build_cloud(cfg["clouds"][0])
    cores = os.cpu_count() or 1
    n = int(min(args.ref_photons, cfg["run"]["n_photons"]))
    ev = 0
    gas = _oracle_gas(cfg, oc)
    for i in range(args.warmup):
        omc.run(oc, dict(cfg["run"], seed=1000 + i), n_photons=n, n_threads=cores, gas=gas)
    t = time.perf_counter()
    for i in range(args.steps):
        ev += int(omc.run(oc, dict(cfg["run"], seed=2000 + i), n_photons=n, n_threads=cores, gas=gas).stats["particle_events"])
    dt = time.perf_counter() - t
    val = ev / dt
    sample = f"unit 0 of {cfg['name']}: {n} histories per step (of {cfg['run']['n_photons']}), {args.steps} steps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True, "scaling": args.scaling,
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "histories_per_step": n, "n_bins": cfg["run"]["n_bins"]},
        "histories_per_s": n * args.steps / dt,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ------------------------------------------------------------------------------------------- ncu capture -> record
def parse_ncu_csv(path: str) -> dict:
    """Metrics of ONE kernel launch from ncu's long csv (`--csv --log-file`: one row per metric) or the wide one
    (`ncu -i x.ncu-rep --page raw --csv`: header, units row, one row per launch)."""
    import csv
    num = lambda text: float(text.replace(",", ""))
    rows = [r for r in csv.reader(open(path, newline="")) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r or "ID" in r)
    hdr, rows = rows[start], rows[start + 1:]
    out: dict = {}
    if "Metric Name" in hdr:
        i_n, i_u, i_v, i_k = hdr.index("Metric Name"), hdr.index("Metric Unit"), hdr.index("Metric Value"), hdr.index("Kernel Name")
        for r in rows:
            if len(r) > i_v and r[i_n] in NCU_METRICS:
                out[NCU_METRICS[r[i_n]]] = num(r[i_v]) * NCU_SCALE.get(r[i_u], 1.0)
                out["kernel"] = r[i_k]
    else:
        units, vals = rows[0], rows[1]
        for name, key in NCU_METRICS.items():
            if name in hdr:
                j = hdr.index(name)
                out[key] = num(vals[j]) * NCU_SCALE.get(units[j], 1.0)
        out["kernel"] = vals[hdr.index("Kernel Name")]
        ratio = "smsp__thread_inst_executed_per_inst_executed.ratio"       # what `--set full` holds instead of the sum
        if "thread_inst_executed" not in out and ratio in hdr and "inst_executed" in out:
            out["thread_inst_executed"] = out["inst_executed"] * num(vals[hdr.index(ratio)])
    missing = [k for k in NCU_REQUIRED if k not in out]
    if missing:
        raise SystemExit(f"{path}: metrics missing: {missing}")
    return out


def ingest_ncu(args):
    """`--ingest-ncu csv --config I`: prints the one-line record of that capture, keyed by the sha256 of the kernel sources."""
    from paper_2012_00963_b200.build import kernel_source_hash
    cfg = _workload(args.config)
    n = int(args.photons or cfg["run"]["n_photons"]) * len(cfg["clouds"]) * len(cfg["t_snap"])
    rec = {"workload": cfg["name"], "histories_per_launch": n, "kernel_source_sha256": kernel_source_hash()}
    rec.update(parse_ncu_csv(args.ingest_ncu))
    for k in ("thread_inst_executed", "inst_executed", "dram_bytes_read", "dram_bytes_write", "smem_wavefronts", "shared_atom_inst"):
        if k in rec:
            rec[k] = int(round(rec[k]))
    rec["lanes_per_inst"] = rec["thread_inst_executed"] / max(rec["inst_executed"], 1)
    rec["command"] = args.command
    print(json.dumps(rec))


# ------------------------------------------------------------------------------------------------------- GPU arm
def _captured_counters(workload: str, histories_per_launch: int):
    """Counters of one transport-kernel launch of this workload from a committed ncu capture (a record written by
    `bench.py --ingest-ncu`), or None when there is none for the kernel sources as they are now."""
    from paper_2012_00963_b200.build import kernel_source_hash
    want = kernel_source_hash()
    found = None
    for path in COUNTERS_FILES:
        if found is not None or not os.path.exists(path):
            continue
        with open(path) as f:
            for line in f:
                line = line.strip()
                if not line.startswith("{"):
                    continue
                rec = json.loads(line)
                if rec.get("workload") == workload and rec.get("histories_per_launch") == histories_per_launch \
                        and rec.get("kernel_source_sha256") == want:
                    found = rec
    return found


def time_workload(P, torch, dist, cfg, args, *, steps, warmup, e2e_steps, rank, world, local, clk, want_peaks=None):
    """Times `steps` steps of workload `cfg` on this rank's GPU (device-resident leg and host-buffer leg); returns the
    measurements reduced over ranks (times: max; counts: sum)."""
    from paper_2012_00963_b200 import _shard
    dev = torch.device("cuda", local)
    if args.depth_model:
        cfg = dict(cfg, clouds=[dict(c, depth_model=args.depth_model) for c in cfg["clouds"]])
    run = dict(cfg["run"])
    n_job = int(args.photons or run["n_photons"])                      # histories per unit of the job (per rank when weak)
    nb, t_all_snaps = run["n_bins"], cfg["t_snap"]
    nc_job, ns_job = len(cfg["clouds"]), len(t_all_snaps)
    # What this rank runs: a list of SEGMENTS, each one pdv_mc_run call over a clouds x snapshots grid with its own id range.
    # One GPU, weak scaling and one-unit jobs: one segment (_shard.plan).  Strong scaling of a multi-unit job: a contiguous stretch
    # of the job's cost line (the library's own flights-per-history estimate), units that straddle a rank boundary split by photon
    # id (_shard.plan_balanced): at most a partial unit at each end and the whole units in between.
    n_units_job = nc_job * ns_job
    if world > 1 and args.scaling == "strong" and n_units_job > 1:
        probe = [P.pdv_cloud_create(c) for c in cfg["clouds"]]             # host optics only matter here (memoised per class)
        costs = [c.estimated_flights(run) for c in probe for _ in t_all_snaps]
        for c in probe:
            c.destroy()
        segs = _shard.plan_balanced(costs, nc_job, ns_job, n_job, rank, world)
        for sg in segs:
            sg["unit_streams"] = sg["unit_ids"]
    else:
        pl = _shard.plan(nc_job, ns_job, n_job, rank, world, args.scaling)
        if world > 1 and args.scaling == "strong":
            pl["unit_streams"] = pl["unit_ids"]
        segs = [pl] if pl["clouds"] and pl["snaps"] else []
    row = 0
    for sg in segs:
        sg["params"] = [cfg["clouds"][i] for i in sg["clouds"]]
        sg["t"] = [t_all_snaps[j] for j in sg["snaps"]]
        sg["run"] = dict(run, first_photon_id=sg["first_photon_id"], **({"unit_streams": sg["unit_streams"]} if "unit_streams" in sg else {}))
        sg["rows"] = (row, row + len(sg["unit_ids"]))
        row += len(sg["unit_ids"])
        sg["handles"] = [P.pdv_cloud_create(c) for c in sg["params"]]
    n_units = row
    unit_ids = [u for sg in segs for u in sg["unit_ids"]]
    hist_per_step = sum(sg["n_photons"] * len(sg["unit_ids"]) for sg in segs)      # histories this rank runs per step
    n = segs[0]["n_photons"] if segs else 0
    photons_job = n_job * (world if args.scaling == "weak" else 1)     # histories per unit of the whole job
    SB = P.STATS_DTYPE.itemsize
    hist = torch.zeros((max(n_units, 1), nb), dtype=torch.float64, device=dev)
    hist2 = torch.zeros_like(hist)
    stats = torch.zeros(max(n_units, 1) * SB, dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2
    stream = torch.cuda.current_stream()
    sweep = "points" in cfg                                   # sweep + interpretation workload: one v_fs per spectrum
    v_fs_job = torch.tensor([c["v_fs"] for c in cfg["clouds"] for _ in t_all_snaps], dtype=torch.float64, device=dev) if sweep else None

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def read_stats():
        return np.frombuffer(stats.cpu().numpy().tobytes(), dtype=P.STATS_DTYPE)[:n_units]

    def step(i):
        ms = 0.0
        for sg in segs:
            a, b = sg["rows"]
            P.pdv_mc_run_device(sg["handles"], sg["t"], sg["n_photons"], run["seed"] + 7919 * i, sg["run"], hist[a:b], hist2[a:b],
                                stats[a * SB:b * SB], stream=stream.cuda_stream)
            if timing[0]:
                ms += P.pdv_last_launch_info()["transport_ms"]       # waits for this segment's kernel (one GPU: the only one)
        if world > 1:                                        # the one exchange: tallies of the whole job on every rank, all on the device
            h, _, _ = _shard.reduce_job(hist[:n_units], hist2[:n_units], stats[:n_units * SB], unit_ids, n_units_job)
        else:
            h = hist[:n_units]
        sp = P.pdv_spectrogram(h, photons_job, run["v_lo"], run["v_hi"], scale=2, stream=stream.cuda_stream)
        if sweep:                                            # row f1: peak position / value / curvature of every spectrum
            sp = P.pdv_spectrum_peaks(h, photons_job, run["v_lo"], run["v_hi"], v_fs_job, half=6, n_pass=2, fit_half=16,
                                      x_min=1.03, stream=stream.cuda_stream)
        return sp, ms

    timing = [False]
    for i in range(warmup):
        flush.zero_()
        step(i)
    barrier()

    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    tot = dict(particle_events=0, surface_reflections=0, histories=0)
    transport_ms = []
    clk.reset()
    timing[0] = world == 1                                   # per-kernel times (roofline) on one GPU only: reading them waits for the kernel
    with clk:                                                # sampled during the device-timed steps and the end-to-end steps
        barrier()
        for i in range(steps):
            flush.zero_()                                    # L2 flush between timed iterations (outside the events)
            ev0[i].record(stream)
            _, ms = step(warmup + i)
            ev1[i].record(stream)
            transport_ms.append(ms)
            s = read_stats()
            for k in tot:
                tot[k] += int(s[k].sum())
        barrier()
    step_ms = sum(a.elapsed_time(b) for a, b in zip(ev0, ev1))
    info = P.pdv_last_launch_info()
    t_all = torch.tensor([step_ms, sum(transport_ms)], dtype=torch.float64, device=dev)
    cnt = torch.tensor([tot["particle_events"], tot["surface_reflections"], tot["histories"]], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t_all, op=dist.ReduceOp.MAX)
        dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    step_ms, tr_ms = (float(x) for x in t_all.cpu())
    events, reflections, histories = (float(x) for x in cnt.cpu())

    # ---- end to end through the host-buffer API (every step: host tables + H2D, run, D2H, spectrogram) ----------------
    # warm: the per-class Mie tables come from the library's memo after the first step; cold: the wavelength moves by
    # 1e-12 per step, so every size parameter is new and every Mie table is computed again
    phase_names = ("cloud_create_ms", "run_ms", "spectrogram_ms")
    v_fs_host = [c["v_fs"] for c in cfg["clouds"] for _ in t_all_snaps]

    def e2e_step(i, phases, cold=0):
        t0 = time.perf_counter()
        cl = [[P.pdv_cloud_create(dict(c, wavelength=c["wavelength"] * (1.0 + 1e-12 * cold)) if cold else c) for c in sg["params"]] for sg in segs]
        t1 = time.perf_counter()
        # a rank without units (strong scaling with fewer units than ranks) only takes part in the reduction
        ev, rh, rh2, rs = 0, [np.zeros((0, nb))], [np.zeros((0, nb))], [np.zeros(0, dtype=P.STATS_DTYPE)]
        for sg, handles in zip(segs, cl):
            r = P.pdv_mc_run(handles, sg["t"], sg["n_photons"], run["seed"] + 104729 * (i + 1), sg["run"])
            ev += int(r.stats["particle_events"].sum())
            rh.append(r.hist.reshape(-1, nb)); rh2.append(r.hist2.reshape(-1, nb)); rs.append(r.stats.reshape(-1))
        rh, rh2, rs = np.concatenate(rh), np.concatenate(rh2), np.concatenate(rs)
        t2 = time.perf_counter()
        if world > 1:
            h, _, _ = _shard.reduce_job(torch.from_numpy(rh).to(dev), torch.from_numpy(rh2).to(dev), rs, unit_ids, n_units_job)
            h = h.cpu().numpy()
        else:
            h = rh
        sp = P.pdv_spectrogram(h, photons_job, run["v_lo"], run["v_hi"], scale=2)
        if sweep:
            sp = P.pdv_spectrum_peaks(h, photons_job, run["v_lo"], run["v_hi"], v_fs_host, half=6, n_pass=2, fit_half=16, x_min=1.03)
        for handles in cl:
            for c in handles:
                c.destroy()
        t3 = time.perf_counter()
        for k, dt in zip(phase_names, (t1 - t0, t2 - t1, t3 - t2)):
            phases[k] = phases.get(k, 0.0) + 1e3 * dt
        return ev, sp

    def e2e_leg(n_steps, cold):
        """-> (events, seconds, phases summed over the steps) of n_steps timed end-to-end steps, max / sum over ranks."""
        phases = {}
        ev = 0
        barrier()
        with clk:
            t0 = time.perf_counter()
            for i in range(n_steps):
                ev += e2e_step(i + (1000 if cold else 0), phases, cold=(1 + i + 7 * _E2E_COLD_CALLS[0]) if cold else 0)[0]
            torch.cuda.synchronize()
            sec = time.perf_counter() - t0
        if cold:
            _E2E_COLD_CALLS[0] += 1
        tt = torch.tensor([sec] + [phases.get(k, 0.0) for k in phase_names], dtype=torch.float64, device=dev)
        cc = torch.tensor([float(ev)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dist.all_reduce(cc, op=dist.ReduceOp.SUM)
        tt = [float(x) for x in tt.cpu()]
        return float(cc), tt[0], {k: v / max(n_steps, 1) for k, v in zip(phase_names, tt[1:])}

    for i in range(2 if e2e_steps else 0):
        e2e_step(-1 - i, {})
    e2e_c, e2e_t, e2e_phases = e2e_leg(e2e_steps, cold=False) if e2e_steps else (0.0, 0.0, {})
    cold_steps = min(e2e_steps, 3)
    cold_c, cold_t, cold_phases = e2e_leg(cold_steps, cold=True) if cold_steps else (0.0, 0.0, {})
    blob_bytes = max(info["smem_bytes"] - 16 * nb, 0)                           # largest cloud image staged per block
    n_handles = sum(len(sg["handles"]) for sg in segs)
    h2d = n_handles * blob_bytes + 24 * n_units + 4 * info["grid"] + 8 * n_units_job * nb   # tables + unit table + block starts + hist (spectrogram)
    d2h = 2 * 8 * n_units * nb + n_units * P.STATS_DTYPE.itemsize + 4 * n_units_job * nb
    for sg in segs:
        for c in sg["handles"]:
            c.destroy()

    out = None
    if rank == 0:
        clocks = clk.summary()
        peaks = want_peaks
        sm_max = clocks["sm_max_mhz"] or 1965.0
        n_sm = peaks["n_sm"]
        issue_peak = n_sm * 4 * 32 * sm_max * 1e6                               # 1 warp-instruction / clk / sub-partition
        a = dict(ALG_INST_PER_FLIGHT)
        if args.depth_model == 1:                      # closed-form v(T): log + 2 FMA (4 with the clamp) instead of the 8 of the table probe
            a["scatter"] -= 4
        if any(c.get("gas_density", 0.0) > 0.0 for c in cfg["clouds"]):
            # gas unit (row f4): class by bisection of the depth bin's 16 thresholds (4 steps x load, compare, add) + per-class albedo
            # and table base (2) + velocity from the closed form of the drag law (multiply, ex2, subtract, multiply, add, select: 6)
            a["scatter"] += 20
        elif any(len(c.get("diameters", [])) > 1 or "lognormal" in c for c in cfg["clouds"]):
            a["scatter"] += 6                        # polydisperse: class pick (guide byte, threshold, compare, clamp) + per-class albedo and table base
        alg = (events * a["scatter"] + reflections * a["reflect"] + histories * a["exit"]) / world
        tr_s = max(tr_ms, 1e-9) * 1e-3
        achieved = alg / tr_s
        cap = _captured_counters(cfg["name"], hist_per_step) if world == 1 else None
        launch_s = tr_s / steps                                                 # one transport-kernel launch, CUDA events, this run
        executed = cap["thread_inst_executed"] / launch_s if cap else None      # executed thread-instructions / s
        roof = {"bound": "alu",
                "achieved": executed / 1e12 if cap else None, "peak": issue_peak / 1e12, "unit": "Tthread-inst/s",
                "frac": executed / issue_peak if cap else None,
                "frac_is": "executed thread-instructions of one launch (ncu capture keyed by the kernel-source sha256, profiles/) / the "
                           "launch duration measured in this run (CUDA events) / peak" if cap else
                           "null: no ncu capture under profiles/ matches the kernel sources as they are (bench.py --ingest-ncu writes one)",
                "traffic": (cap["dram_bytes_read"] + cap["dram_bytes_write"]) if cap else None,
                "traffic_is": "dram bytes of one launch (same capture)" if cap else "no capture",
                "executed_thread_inst_per_launch": cap["thread_inst_executed"] if cap else None,
                "frac_of_measured_ffma": executed / peaks["ffma_thread_inst_per_s"] if cap else None,
                "peak_is": f"{n_sm} SMs x 4 sub-partitions x 32 lanes x {sm_max:.0f} MHz (DESIGN.md), not in MEASURED_PEAKS.json",
                "kernel": "pdv::transport_kernel",
                "measured_ffma_Tinst_s": peaks["ffma_thread_inst_per_s"] / 1e12,
                "measured_mufu_Tinst_s": peaks["mufu_thread_inst_per_s"] / 1e12,
                "sm_clock_mhz_in_microbench": peaks["sm_clock_mhz"],
                "frac_model": achieved / issue_peak, "achieved_model": achieved / 1e12, "alg_inst_per_flight": a,
                "frac_model_is": "hand count of algorithmic instructions per flight x flights / time / peak: charges every flight a whole "
                                 "Philox block, so it EXCEEDS the executed count; context only"}
        for k in ("lanes_per_inst", "issue_active_pct", "pipe_alu_pct", "pipe_fmaheavy_pct", "pipe_xu_pct", "smem_wavefronts_pct",
                  "warps_active_pct", "shared_atom_inst"):
            roof[k] = cap.get(k) if cap else None
        out = {
            "value": events / (step_ms * 1e-3), "ms_per_step": step_ms / steps, "steps": steps, "warmup": warmup,
            "config": {"workload": cfg["name"], "histories_per_step_per_gpu": hist_per_step, "units": n_units_job, "depth_model": args.depth_model,
                       "n_bins": nb, "parallelism": f"{args.scaling}: " + ("photon-id ranges" if args.scaling == "weak" or n_units_job == 1 else "equal estimated cost (units split by photon id at rank boundaries)") + f" x{world}",
                       "l2": "flushed between steps (256 MiB write)",
                       "events_per_history": events / max(histories, 1), "reflections_per_history": reflections / max(histories, 1)},
            "histories_per_s": histories / (step_ms * 1e-3),
            "events_incl_surface_per_s": (events + reflections) / (step_ms * 1e-3),
            "gpu_launches": (2 * max(len(segs), 1) + (2 if sweep else 1)) * steps,    # (transport + finalize) per segment + spectrogram (+ peak) kernels per step
            "launch": {"grid": info["grid"], "block": info["block"], "smem_bytes": info["smem_bytes"],
                       "transport_ms_per_step": tr_ms / steps},
            "clocks": clocks,
            "e2e": {"value": (e2e_c / e2e_t) if e2e_steps else None, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "steps": e2e_steps, "ms_per_step": (1e3 * e2e_t / e2e_steps) if e2e_steps else None,
                    "includes": "pdv_cloud_create (host tables + H2D; per-class Mie tables from the library's memo: WARM after the "
                                "first step), pdv_mc_run (host outputs), pdv_spectrogram" + (", pdv_spectrum_peaks" if sweep else ""),
                    "phases": e2e_phases,
                    "cold": {"value": (cold_c / cold_t) if cold_steps else None, "ms_per_step": (1e3 * cold_t / cold_steps) if cold_steps else None,
                             "steps": cold_steps, "phases": cold_phases,
                             "is": "the same step with the Mie memo defeated (wavelength x (1 + k 1e-12), a new k per step): "
                                   "every per-class Mie table is computed again on the host"}},
            "roofline": roof,
        }
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1,
                    help="BASELINE.json configs index (default 1 = headline); 5 = the paper's Figs. 13-15 sweep (SURVEY.md 8(f) row "
                         "f1: 14 clouds x 1e7 photons in one launch, then pdv_spectrum_peaks on the device); 6 = row f4: a 16-class cloud "
                         "in a gas environment, 20 snapshots x 1e7 photons")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"], help="N > 1: how the job is shared (see the module docstring)")
    ap.add_argument("--photons", type=int, default=0, help="override histories per unit (debugging; invalidates the number)")
    ap.add_argument("--depth-model", type=int, default=0, choices=[0, 1],
                    help="0: depth table (the headline design); 1: closed-form v(T), exponential profiles only (variant f2)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--ref-photons", type=int, default=2_000_000, help="--impl reference: histories per step")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="CPU work of the cpu_baseline leg (0: skip)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps of the host-buffer leg (0: same as --steps)")
    ap.add_argument("--other-configs", type=int, default=-1,
                    help="1: append the 'configs' array (the other workloads at full size, 2 timed steps each); 0: skip; "
                         "default: 1 for the plain default run on one GPU (no --config), else 0")
    ap.add_argument("--other-cpu-seconds", type=float, default=1.5, help="CPU work of the cpu_baseline of each entry of 'configs'")
    ap.add_argument("--ingest-ncu", default="", metavar="CSV",
                    help="no GPU work: turn the ncu csv of ONE transport-kernel launch of --config (and --photons) into the record that "
                         "roofline.frac is computed from; append the printed line to profiles/r3_transport_counters.txt")
    ap.add_argument("--command", default="", help="--ingest-ncu: the full ncu command that wrote the csv")
    args = ap.parse_args()
    if args.ingest_ncu:
        ingest_ncu(args)
        return
    if args.impl == "reference":
        run_reference(args)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist

    import paper_2012_00963_b200 as P

    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    clk = ClockSampler(local, str(getattr(torch.cuda.get_device_properties(local), "uuid", "")))
    peaks = P.pdv_issue_peaks(30.0) if rank == 0 else None

    cfg = _workload(args.config)
    main_out = time_workload(P, torch, dist, cfg, args, steps=args.steps, warmup=args.warmup, e2e_steps=args.e2e_steps or args.steps,
                             rank=rank, world=world, local=local, clk=clk, want_peaks=peaks)
    others = []
    do_others = args.other_configs == 1 or (args.other_configs < 0 and world == 1 and args.config == 1 and not args.depth_model)
    if do_others:
        for idx in (0, 2, 3, 4, 5, 6):
            if idx == args.config:
                continue
            wl = _workload(idx)
            o = time_workload(P, torch, dist, wl, args, steps=2, warmup=3, e2e_steps=2, rank=rank, world=world, local=local,
                              clk=clk, want_peaks=peaks)
            if o is not None:
                others.append({"workload": o["config"]["workload"], "config_index": idx, "value": o["value"], "unit": UNIT,
                               "ms_per_step": o["ms_per_step"], "steps": o["steps"], "warmup": o["warmup"],
                               "histories_per_s": o["histories_per_s"], "transport_ms_per_step": o["launch"]["transport_ms_per_step"],
                               "launch": o["launch"], "config": o["config"], "gpu_launches": o["gpu_launches"],
                               "e2e": {k: o["e2e"][k] for k in ("value", "ms_per_step", "phases", "cold")},
                               "roofline": {k: o["roofline"][k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic",
                                                                          "executed_thread_inst_per_launch", "frac_of_measured_ffma",
                                                                          "frac_model", "lanes_per_inst", "issue_active_pct", "pipe_alu_pct",
                                                                          "pipe_fmaheavy_pct", "pipe_xu_pct", "smem_wavefronts_pct")},
                               "clocks": o["clocks"]})
                if args.other_cpu_seconds > 0:
                    others[-1]["cpu_baseline"] = _cpu_baseline(wl, args.other_cpu_seconds, seed=97 + idx)
    if rank == 0:
        out = {"metric": METRIC, "value": main_out["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
               "ms_per_step": main_out["ms_per_step"], "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
               "dtype": "f32", "data": "synthetic"}
        out.update({k: main_out[k] for k in ("config", "histories_per_s", "events_incl_surface_per_s", "gpu_launches", "launch", "clocks",
                                             "e2e", "roofline")})
        if args.cpu_seconds > 0:
            out["cpu_baseline"] = _cpu_baseline(cfg, args.cpu_seconds, seed=97)
        if others:
            out["configs"] = others
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
