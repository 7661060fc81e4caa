"""bench.py's reference arm runs on CPU (it times the oracle): check the JSON-line contract the
driver parses, and the helper arithmetic of the link fractions.  The CUDA arm needs a GPU and is
exercised by the driver / gpurun."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--steps", "3", "--warmup", "1", "--scale", "64"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "kv_migration_GBps" and d["unit"] == "GB/s"
    assert d["steps"] == 3 and d["warmup"] == 1 and d["n_gpus"] == 1 and d["higher_is_better"] is True
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"] and d["config"]["scale"] == 64
    assert d["cpu_baseline"]["cores"] == 1 and d["cpu_baseline"]["cpu_model"]


def test_reference_arm_f_busy_and_threads():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "3",
                        "--f-busy", "0.75", "--steps", "6", "--warmup", "3", "--scale", "128", "--ref-threads", "2"],
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads(r.stdout.strip())
    assert "f0.75" in d["config"]["workload"] and d["cpu_baseline"]["cores"] == 2 and d["value"] > 0


def test_cpu_baseline_reports_one_core_and_all_cores():
    sys.path.insert(0, ROOT)
    import bench
    cb = bench.cpu_baseline(2, budget_s=1.0, scale=64)
    assert cb["cores"] == 1 and cb["value"] > 0 and cb["kind"] == "oracle"
    assert cb["all_cores"]["cores"] == os.cpu_count() and cb["all_cores"]["value"] > 0
    assert cb["cpu_model"] and cb["scale"] == 64


def test_non_zero_ranks_of_the_reference_arm_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_link_bounds():
    sys.path.insert(0, ROOT)
    import bench
    link = {"d2h": 57.2, "h2d": 55.6, "bidir_sum": 99.8}
    G = 2 ** 30
    # one direction only: bound = model = bytes / solo rate
    assert np.isclose(bench.ideal_seconds(5 * G, 0, link), 5 * G / 57.2e9)
    assert np.isclose(bench.memcpy_model_seconds(5 * G, 0, link), 5 * G / 57.2e9)
    assert np.isclose(bench.memcpy_model_seconds(0, 5 * G, link), 5 * G / 55.6e9)
    # the model is never below the bound, and equals it when both directions end together
    for d, p in ((10.2, 3.64), (1, 1), (0.1, 7), (3, 3.1)):
        assert bench.memcpy_model_seconds(d * G, p * G, link) >= bench.ideal_seconds(d * G, p * G, link) * (1 - 1e-12)
    d = 57.2 / (57.2 + 55.6) * 10 * G; p = 55.6 / (57.2 + 55.6) * 10 * G
    assert np.isclose(bench.memcpy_model_seconds(d, p, link), 10 * G / 99.8e9)


def test_roofline_traffic_comes_from_a_tracked_ncu_summary():
    """bench.py prints `roofline.traffic` from profiles/ncu_traffic.json (no constant in the code): the
    file must name its source capture and launch, and its ratio must be read + write over 2 x bytes."""
    sys.path.insert(0, ROOT)
    import bench
    t = bench._load_ncu_traffic()
    for k in ("dram_bytes_per_launch", "dram_bytes_read", "dram_bytes_write", "algorithmic_bytes_same_launch",
              "ratio", "launch", "source", "kernel"):
        assert k in t, k
    assert np.isclose(t["dram_bytes_per_launch"], t["dram_bytes_read"] + t["dram_bytes_write"])
    assert np.isclose(t["ratio"], t["dram_bytes_per_launch"] / t["algorithmic_bytes_same_launch"], atol=5e-4)
    assert 0.9 < t["ratio"] < 1.1
    assert os.path.exists(os.path.join(ROOT, t["source"].split(" ")[0]))
