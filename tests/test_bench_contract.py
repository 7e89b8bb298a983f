"""The driver's contract with bench.py: ONE JSON line on stdout with the keys the brief names.  The reference arm (the CPU
oracle on host cores) runs without a GPU; the llx arm is a `-m gpu` test."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
             "dtype", "data", "config", "e2e", "gpu_launches", "cpu_baseline"}


def run_bench(*args, timeout=900):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=timeout, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, f"bench.py must print ONE line, got {len(lines)}"
    return json.loads(lines[0])


def test_reference_arm_prints_the_contract_line_without_a_gpu():
    d = run_bench("--impl", "reference", "--steps", "2", "--warmup", "1")
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["metric"] == "kv_migration_gbps_rd_plus_wr" and d["unit"] == "GB/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["gpu_launches"] == 0 and d["vs_baseline"] is None
    assert d["config"]["workload"] == "llama7b_2048tok_3stage_112_14_2"
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["sample"] and cb["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


@pytest.mark.gpu
def test_llx_arm_prints_the_contract_line_with_roofline_e2e_and_clocks():
    d = run_bench("--steps", "30", "--warmup", "3", "--downtime-reps", "10")
    assert BASE_KEYS | {"roofline", "clocks"} <= set(d) and "impl" not in d
    assert d["metric"] == "kv_migration_gbps_rd_plus_wr" and d["dtype"] == "u16" and d["data"] == "synthetic" and d["scaling"] == "weak"
    assert d["n_gpus"] == 1 and d["steps"] == 30 and d["warmup"] == 3 and d["vs_baseline"] is None
    assert d["config"]["workload"] == "llama7b_2048tok_3stage_112_14_2" and "model" not in d["config"]
    # value is bytes of one whole step / time of one whole step; five llx launches per step (3 stages + 2 appends)
    assert abs(d["value"] - 2147483648 / (d["ms_per_step"] * 1e-3) / 1e9) < 1e-6 * d["value"]
    assert d["gpu_launches"] == 5 * 30
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert r["algorithmic_bytes_per_launch"] == 1879048192 and (r["traffic"] is None or 0.5 < r["traffic"] / 1879048192 < 1.2)
    assert 0.5 < r["frac"] < 1.1 and d["value"] < 1.05 * r["peak"]
    e = d["e2e"]
    assert e["unit"] == "GB/s" and e["h2d_bytes_per_step"] == e["d2h_bytes_per_step"] == 1 << 30 and 0 < e["value"] < 0.2 * d["value"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and 0 < cb["value"] < d["value"]
    assert cb["attention_oracle"]["ms"] > 0                                  # a timed sample, not a sentence
    # every BASELINE.json config and both halves of the metric are in the ONE line ("do this" item 1)
    cf = r["configs"]
    assert [x["tokens"] for x in cf["configs2_length_sweep_llama7b"]] == [256, 512, 1024, 2048, 4096, 8192]
    assert all(x["single_shot_GBps"] > 1000 and 0 < x["final_stage_gpu_us_cold"] < 100 for x in cf["configs2_length_sweep_llama7b"])
    assert all(v.get("one_launch_GBps", 0) > 1000 or "skipped" in v for v in cf["configs3_batch_llama30b_64req"].values())
    c4 = cf["configs4_interference_decode_batch32"]
    assert "skipped" in c4 or ([c["budget_GBps"] for c in c4["cases"]] == [0, 25, 12] and c4["decode_step_alone_ms"] > 0)
    assert {"torch_contiguous_copy_GBps", "per_tile_memcpy_loop_GBps"} <= set(cf["reference_points_2048tok_GBps"])
    assert r["downtime_us"]["host_median"] > 0 and r["downtime_us"]["gpu_median"] > 0
    lp = e["link_peak_gbs"]
    assert lp["d2h_GBps"] > 10 and lp["h2d_GBps"] > 10 and 0.3 < e["frac_of_link_duplex"] < 1.05
    v1 = d["value_round1_definition"]
    assert 0.8 * d["value"] < v1["value"] <= 1.02 * d["value"]
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])
    assert not {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"} & set(d["clocks"]["reasons"])
