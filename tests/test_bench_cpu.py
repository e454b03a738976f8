"""CPU checks of bench.py's host logic: the reference arm's JSON line, and that every roofline.traffic figure is read from a
committed ncu raw page (profiles/traffic.json names the file it was extracted from)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_traffic_figures_come_from_committed_ncu_rows():
    import bench
    with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
        table = json.load(f)
    assert {"mid", "long", "adaptive", "dense-equivalence"} <= set(table)
    for workload, entry in table.items():
        path = os.path.join(ROOT, "profiles", entry["source"])
        assert os.path.exists(path), path
        rows = {r.split(",")[0].strip('"'): r for r in open(path).read().splitlines()}
        assert "dram__bytes_read.sum" in rows and "dram__bytes_write.sum" in rows and "gpu__time_duration.sum" in rows
        got, src = bench.ncu_traffic(workload)
        assert got == entry["dram_bytes"] and src == "profiles/" + entry["source"]
    assert bench.ncu_traffic("no-such-workload") == (None, None)
    # every raw page names its command in r2_ncu.md
    md = open(os.path.join(ROOT, "profiles", "r2_ncu.md")).read()
    assert "ncu --set full --clock-control none" in md and "bench.py" in md


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, cwd=ROOT, timeout=300)
    assert out.returncode == 0, out.stderr[-500:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in line, key
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["gpu_launches"] == 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"] and line["value"] > 0
