"""Turns an ncu export of ONE transport-kernel launch into the one-line record that bench.py reads.

    ncu --metrics smsp__thread_inst_executed.sum,smsp__inst_executed.sum,dram__bytes_read.sum,dram__bytes_write.sum,gpu__time_duration.sum \\
        --clock-control none -k regex:transport_kernel -s 3 -c 1 --csv --log-file gpurun_out/counters_cfg2.csv \\
        python bench.py --config 1 --steps 1 --warmup 3 --cpu-seconds 0 --e2e-steps 1 --other-configs 0
    python -m paper_2012_00963_b200.ncu_counters gpurun_out/counters_cfg2.csv --config 1 --command "<the ncu command>" \\
        >> profiles/r2_transport_counters.txt

Accepts ncu's long CSV (one row per metric, `--csv --log-file`) and the wide one (`ncu -i x.ncu-rep --page raw --csv`).
The record carries the sha256 of the kernel sources (build.kernel_source_hash): bench.py prints `roofline.traffic` (dram bytes of
the launch) and `roofline.frac_executed` (executed thread-instructions / time / issue peak) only from a record whose key
matches the sources it runs, so a capture can never go stale silently.  Nothing of the method's arithmetic lives here.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WANT = {"smsp__thread_inst_executed.sum": "thread_inst_executed", "smsp__inst_executed.sum": "inst_executed",
        "dram__bytes_read.sum": "dram_bytes_read", "dram__bytes_write.sum": "dram_bytes_write",
        "gpu__time_duration.sum": "gpu_time_ms"}
SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1e-6, "us": 1e-3, "usecond": 1e-3, "ms": 1.0, "msecond": 1.0,
         "nsecond": 1e-6, "second": 1e3, "s": 1e3, "inst": 1.0, "": 1.0}


def _num(text: str) -> float:
    return float(text.replace(",", ""))


def parse(path: str) -> dict:
    rows = [r for r in csv.reader(open(path, newline="")) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r or "ID" in r)
    hdr, rows = rows[start], rows[start + 1:]
    out: dict = {}
    if "Metric Name" in hdr:                                   # long format
        i_n, i_u, i_v, i_k = hdr.index("Metric Name"), hdr.index("Metric Unit"), hdr.index("Metric Value"), hdr.index("Kernel Name")
        for r in rows:
            if len(r) > i_v and r[i_n] in WANT:
                out[WANT[r[i_n]]] = _num(r[i_v]) * SCALE.get(r[i_u], 1.0)
                out["kernel"] = r[i_k]
    else:                                                      # wide format: header, units row, one row per launch
        units, vals = rows[0], rows[1]
        for name, key in WANT.items():
            if name in hdr:
                j = hdr.index(name)
                out[key] = _num(vals[j]) * SCALE.get(units[j], 1.0)
        out["kernel"] = vals[hdr.index("Kernel Name")]
        ratio = "smsp__thread_inst_executed_per_inst_executed.ratio"       # what `--set full` holds instead of the sum
        if "thread_inst_executed" not in out and ratio in hdr and "inst_executed" in out:
            out["thread_inst_executed"] = out["inst_executed"] * _num(vals[hdr.index(ratio)])
    missing = [k for k in WANT.values() if k not in out]
    if missing:
        raise SystemExit(f"{path}: metrics missing: {missing}")
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("csv")
    ap.add_argument("--config", type=int, required=True, help="bench.py --config index of the captured workload")
    ap.add_argument("--photons", type=int, default=0, help="histories per unit if the capture overrode them")
    ap.add_argument("--command", default="", help="the full ncu command that wrote the csv")
    a = ap.parse_args()
    import bench
    from paper_2012_00963_b200.build import kernel_source_hash
    cfg = bench._workload(a.config)
    n = (a.photons or cfg["run"]["n_photons"]) * len(cfg["clouds"]) * len(cfg["t_snap"])
    rec = {"workload": cfg["name"], "histories_per_launch": n, "kernel_source_sha256": kernel_source_hash()}
    rec.update(parse(a.csv))
    for k in ("thread_inst_executed", "inst_executed", "dram_bytes_read", "dram_bytes_write"):
        rec[k] = int(round(rec[k]))
    rec["lanes_per_inst"] = rec["thread_inst_executed"] / max(rec["inst_executed"], 1)
    rec["command"] = a.command
    print(json.dumps(rec))


if __name__ == "__main__":
    main()
