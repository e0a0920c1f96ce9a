"""bench.py prints ONE JSON line with the keys the driver reads (task contract).

CPU: the reference arm (the oracle timed on the host cores) on the reduced configs. GPU: the product arm on a reduced
config, checked for the same keys plus roofline / e2e / gpu_launches / clocks.
"""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
             "dtype", "data", "config", "e2e", "cpu_baseline"}


def run_bench(*argv, env=None):
    e = dict(os.environ)
    e.update(env or {})
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], cwd=ROOT, env=e, capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    return [l for l in p.stdout.splitlines() if l.strip()]


@pytest.mark.parametrize("config,sampler", [("c1", "exp"), ("c4", "exp"), ("c3", "poisson")])
def test_reference_arm_line(config, sampler):
    lines = run_bench("--impl", "reference", "--small", "--config", config, "--sampler", sampler, "--steps", "1", "--warmup", "0")
    assert len(lines) == 1
    r = json.loads(lines[0])
    assert BASE_KEYS <= set(r)
    assert r["impl"] == "reference" and r["metric"] == "lineage_events_per_s" and r["unit"] == "events/s"
    assert r["higher_is_better"] is True and r["vs_baseline"] is None and r["data"] == "synthetic"
    assert r["value"] > 0 and r["ms_per_step"] > 0
    assert r["config"]["event_time_sampler"] == sampler and "workload" in r["config"]
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["cores"] == 1 and r["cpu_baseline"]["value"] == r["value"]
    assert r["e2e"] == {"value": r["value"], "unit": r["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_do_no_work():
    # under torchrun only rank 0 runs and prints the oracle line
    assert run_bench("--impl", "reference", "--small", "--config", "c1", "--gpus", "2", env={"RANK": "1", "WORLD_SIZE": "2"}) == []


@pytest.mark.gpu
@pytest.mark.parametrize("config,sampler", [("c4", "exp"), ("c2", "poisson")])
def test_product_arm_line(config, sampler):
    lines = run_bench("--small", "--config", config, "--sampler", sampler, "--steps", "2", "--warmup", "3")
    assert len(lines) == 1
    r = json.loads(lines[0])
    assert BASE_KEYS | {"roofline", "clocks", "gpu_launches"} <= set(r)
    assert "impl" not in r or r["impl"] == "ours"
    assert r["n_gpus"] == 1 and r["steps"] == 2 and r["warmup"] == 3 and r["scaling"] == "weak" and r["dtype"] == "int64"
    assert r["value"] > 0 and r["gpu_launches"] > 0
    e = r["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] >= 0 and e["d2h_bytes_per_step"] > 0 and e["value"] != r["value"]
    rf = r["roofline"]
    assert rf["bound"] == "alu" and rf["peak"] > 0 and rf["achieved"] > 0 and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(r["clocks"])
    cb = r["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["value"] > 0 and cb["cores"] == 1 and cb["sample"]


@pytest.mark.gpu
def test_product_arm_event_stream_leg():
    """--event-stream adds the step timed with the full event stream recorded to the same line."""
    lines = run_bench("--small", "--config", "c4", "--event-stream", "22", "--steps", "1", "--warmup", "3", "--no-cpu-baseline")
    assert len(lines) == 1
    r = json.loads(lines[0])
    s = r["event_stream"]
    assert s["ms_per_step"] > 0 and s["distinct_events"] >= r["richness"] > 0 and s["distinct_events_per_s"] > 0 and s["epochs"] >= 1


@pytest.mark.gpu
def test_product_arm_partitioned_mode():
    """--mode partitioned drives dist.simulate_partitioned (isolated partitions + merge) and prints the same line shape."""
    lines = run_bench("--small", "--config", "c4", "--mode", "partitioned", "--steps", "2", "--warmup", "3")
    assert len(lines) == 1
    r = json.loads(lines[0])
    assert r["config"]["parallelism"] == "partitions x1" and r["scaling"] == "strong" and r["n_gpus"] == 1
    assert r["value"] > 0 and r["gpu_launches"] > 0 and r["merge"]["ms_per_step"] > 0 and r["richness"] > 0
