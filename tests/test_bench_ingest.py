"""CPU: bench.py --ingest-ncu turns the ncu csv of one transport-kernel launch into the record roofline.frac is computed from
(host logic only; the csv below is a hand-made export in ncu's long format, not a measurement)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CSV = '''==PROF== Connected to process 1
"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"
"0","1","python","h","void pdv::transport_kernel<0>(pdv::RunParams)","1","7","(1024, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","dram__bytes_read.sum","Kbyte","66.5"
"0","1","python","h","void pdv::transport_kernel<0>(pdv::RunParams)","1","7","(1024, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","dram__bytes_write.sum","byte","0"
"0","1","python","h","void pdv::transport_kernel<0>(pdv::RunParams)","1","7","(1024, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","gpu__time_duration.sum","us","3,300.5"
"0","1","python","h","void pdv::transport_kernel<0>(pdv::RunParams)","1","7","(1024, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","smsp__inst_executed.sum","inst","1,000"
"0","1","python","h","void pdv::transport_kernel<0>(pdv::RunParams)","1","7","(1024, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","smsp__thread_inst_executed.sum","inst","24,000"
"0","1","python","h","void pdv::transport_kernel<0>(pdv::RunParams)","1","7","(1024, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","smsp__issue_active.avg.pct_of_peak_sustained_active","%","78.5"
'''


def test_ingest_long_csv(tmp_path):
    from paper_2012_00963_b200.build import kernel_source_hash
    f = tmp_path / "c.csv"
    f.write_text(CSV)
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--ingest-ncu", str(f), "--config", "1", "--command", "ncu ..."],
                         cwd=ROOT, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stderr[-1000:]
    rec = json.loads(out.stdout.strip())
    assert rec["workload"] == "cfg2_multi_mono" and rec["histories_per_launch"] == 10 ** 8
    assert rec["kernel_source_sha256"] == kernel_source_hash() and rec["command"] == "ncu ..."
    assert rec["thread_inst_executed"] == 24000 and rec["inst_executed"] == 1000 and rec["lanes_per_inst"] == 24.0
    assert rec["dram_bytes_read"] == 66500 and rec["dram_bytes_write"] == 0 and abs(rec["gpu_time_ms"] - 3.3005) < 1e-9
    assert rec["issue_active_pct"] == 78.5 and "pipe_alu_pct" not in rec


def test_ingest_refuses_a_csv_without_the_required_metrics(tmp_path):
    f = tmp_path / "c.csv"
    f.write_text("\n".join(CSV.splitlines()[:4]) + "\n")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--ingest-ncu", str(f), "--config", "1"],
                         cwd=ROOT, capture_output=True, text=True, timeout=120)
    assert out.returncode != 0 and "metrics missing" in (out.stderr + out.stdout)
