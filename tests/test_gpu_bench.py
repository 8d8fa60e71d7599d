"""GPU: bench.py keeps its contract -- one JSON line with the keys the driver reads (a short run with few photons)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("_library_is_built")]
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("flags", [[], ["--config", "5"]])
def test_bench_prints_one_json_line_with_the_contract_keys(flags):
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--photons", "200000", "--steps", "2", "--warmup", "3",
           "--cpu-seconds", "0.5", "--e2e-steps", "1"] + flags
    out = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["value"] > 0 and "workload" in d["config"] and d["data"] == "synthetic"
    assert d["gpu_launches"] == (4 if flags else 3) * 2
    assert set(("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")) <= set(d["e2e"]) and d["e2e"]["value"] > 0
    assert set(("bound", "achieved", "peak", "unit", "frac", "traffic")) <= set(d["roofline"]) and d["roofline"]["bound"] == "alu"
    assert set(("frac_model", "frac_is", "issue_active_pct", "lanes_per_inst", "smem_wavefronts_pct")) <= set(d["roofline"])
    assert d["roofline"]["frac"] is None or 0.0 < d["roofline"]["frac"] < 1.0           # measured or null, never the model
    assert set(("cloud_create_ms", "run_ms", "spectrogram_ms")) <= set(d["e2e"]["phases"]) and d["e2e"]["cold"]["value"] > 0
    assert d["e2e"]["cold"]["phases"]["cloud_create_ms"] >= d["e2e"]["phases"]["cloud_create_ms"] * 0.5
    assert set(("value", "unit", "cores", "kind", "sample")) <= set(d["cpu_baseline"]) and d["cpu_baseline"]["kind"] == "oracle"
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(d["clocks"])


def test_reference_arm_prints_the_same_shape():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1",
           "--ref-photons", "50000"]
    out = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.strip()][-1])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["config"]["workload"] == "cfg2_multi_mono"
