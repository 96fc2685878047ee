"""bench.py prints ONE JSON line with the keys the driver reads (run on a reduced zone
count so that it takes seconds; the metric itself is quoted at the default 16384 zones)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], cwd=ROOT,
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


@pytest.mark.gpu
def test_bench_line_has_the_contract_keys():
    d = run_bench("--zones", "1024", "--steps", "2", "--warmup", "1", "--no-extra")
    assert d["metric"].startswith("zone-networks integrated per second") and d["unit"] == "zone-networks/s"
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1 and d["higher_is_better"] is True
    assert d["scaling"] == "weak" and d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] == 6  # 2 order kernels + the zone kernel per step
    assert d["ms_per_step_best"] <= d["ms_per_step_median"] and d["value_best"] >= d["value_median"] > 0
    h = d["config"]["sub_steps_per_zone"]
    assert 1 <= h["min"] <= h["median"] <= h["p99"] <= h["max"]
    assert "workload" in d["config"] and "model" not in d["config"]
    r = d["roofline"]
    assert r["bound"] in ("alu", "hbm", "tensor") and r["unit"] == "Tinstr/s" and 0 < r["frac"] < 1
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["traffic"] is None  # not the default workload
    assert 0 < d["roofline_smem"]["frac"] < 1
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 1024 * (150 * 8 + 24) and e["d2h_bytes_per_step"] > 0
    assert e["value"] <= d["value"] * 1.05  # the link inside the timed region: never faster than resident
    assert 0 < e["staged"]["value"] <= d["value"] * 1.05
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]
    assert d["cpu_baseline_1core"]["cores"] == 1 and d["cpu_baseline_1core"]["value"] > 0
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])


@pytest.mark.gpu
def test_reference_arm_times_the_oracle():
    d = run_bench("--impl", "reference", "--steps", "1", "--warmup", "0")
    assert d["impl"] == "reference" and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["e2e"]["value"] == d["value"]


def test_reference_arm_does_not_load_the_product_library():
    """The oracle arm must not map libkinnet.so into its process: import what it
    imports, in a fresh interpreter, and look at the loaded objects."""
    code = ("import sys; sys.argv=['bench.py']; import bench; bench.workload(0, 1, 64); "
            "import oracle; oracle.max_threads(); "
            "maps=open('/proc/self/maps').read(); "
            "assert 'libasym_oracle.so' in maps; assert 'libkinnet' not in maps, 'product library loaded'; "
            "assert 'paper_1409_5826_b200' not in sys.modules")
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
