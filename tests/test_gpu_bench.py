"""bench.py's JSON contract on a small workload (the driver runs the default one): one line, the required keys, launch
count = 4 per step, roofline / e2e / clocks objects; the z-slab decomposition as a 1-rank job."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "20", "--warmup", "3", "--no-cpu-baseline",
                        "--e2e-steps", "2"] + list(extra), capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.strip().splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


@pytest.mark.parametrize("workload,decomp", [("cfg1", "replicas"), ("cfg2", "replicas"), ("cfg2", "slab")])
def test_bench_json_contract(workload, decomp):
    d = _run("--workload", workload, "--decomp", decomp)
    assert d["metric"].startswith("(z,v) cell-updates/sec") and d["unit"] == "cell-updates/s"
    assert d["n_gpus"] == 1 and d["steps"] == 20 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None and d["scaling"] == "weak"
    assert d["value"] > 0 and abs(d["value"] - d["config"]["nz"] * d["config"]["nv"] / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    assert d["config"]["workload"] == workload and "model" not in d["config"]
    assert d["gpu_launches"] == 4 * 20
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] > 1000 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert len(r["per_stage"]) == 4 and r["bytes_per_cell_step"] == 768 and 0.5 < r["stage_kernel_share_of_step"] <= 1.05
    assert r["alu"]["frac"] > 0 and r["survey_model_1024B"]["GBps"] > 0
    e = d["e2e"]
    nbytes = 64 * d["config"]["nz"] * d["config"]["nv"]
    assert e["h2d_bytes_per_step"] == nbytes and e["d2h_bytes_per_step"] == nbytes and 0 < e["value"] < d["value"]
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(d["clocks"])
    assert d["graph_replay"]["value"] > 0
    c = d["checks"]
    assert c["steps_total"] == 3 + 20 + 20                       # warm-up, timed, event-free (graph) pass
    if workload != "cfg1":      # z-homogeneous start without the vacuum term: trace per cell and M0 stay put
        assert c["trace_dev_max"] < 1e-12 and c["dM0_max"] < 1e-8
    if decomp == "slab":
        assert "z-slabs x1" in d["config"]["parallelism"]
