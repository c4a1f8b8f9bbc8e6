"""CPU test of bench.py's reference arm (--impl reference): the one JSON line and its contract keys.
(The CUDA arm needs a GPU; its line is checked by the driver and kept under profiles/.)"""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_contract_line():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg0",
                        "--steps", "2", "--warmup", "3"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "us_per_image_pair" and d["unit"] == "us/pair"
    assert d["higher_is_better"] is False and d["value"] > 0 and d["steps"] == 2 and d["warmup"] == 3
    assert d["config"]["workload"].startswith("cfg0") and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["cpu_baseline"]["value"] == d["value"] and d["e2e"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    # `config` is the GPU arm's, key for key (the driver compares the two); the reference arm's own bounded sample is
    # described in cpu_baseline.sample
    sys.path.insert(0, ROOT)
    import bench
    from paper_2501_10653_b200 import synth
    idx, pairs, _ = bench.WORKLOADS["cfg0"]
    assert d["config"] == bench.workload_config(synth.CONFIGS[idx], pairs, bench.l2_note(synth.CONFIGS[idx], pairs))
    assert "pair(s)" in d["cpu_baseline"]["sample"]


def test_traffic_table_is_machine_written_and_parses():
    """roofline.traffic comes from profiles/ncu_traffic.csv (rows copied out of .ncu-rep files by `bench.py
    --traffic-extract`), keyed by workload, batch size and library version."""
    import csv
    sys.path.insert(0, ROOT)
    import bench
    path = os.path.join(ROOT, bench.NCU_TRAFFIC_FILE)
    assert os.path.exists(path)
    rows = list(csv.DictReader(open(path, newline="")))
    assert rows and list(rows[0].keys()) == bench.TRAFFIC_COLUMNS
    for r in rows:
        total, src = bench.ncu_traffic(r["workload"], int(r["pairs_per_launch"]), r["library_version"])
        assert total == float(r["dram__bytes_read.sum"]) + float(r["dram__bytes_write.sum"]) and r["report"] in src
        assert bench.ncu_traffic(r["workload"], int(r["pairs_per_launch"]), "0.0.0")[0] is None     # another version
    assert bench.ncu_traffic("no_such_workload", 1, "0.0.0")[0] is None


def test_reference_arm_other_ranks_print_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg0",
                        "--steps", "1", "--warmup", "3", "--gpus", "2"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
