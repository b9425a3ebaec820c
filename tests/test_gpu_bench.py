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
                        "--e2e-steps", "2"] + (list(extra) if "--steps" in extra else ["--no-secondary"] + list(extra)),
                       capture_output=True, text=True, timeout=600)
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
    assert r["bound"] in ("hbm", "alu") and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert r["hbm"]["unit"] == "GB/s" and r["hbm"]["peak"] > 1000 and abs(r["hbm"]["frac"] - r["hbm"]["achieved"] / r["hbm"]["peak"]) < 1e-12
    if r["bound"] == "hbm":
        assert r["unit"] == "GB/s" and r["achieved"] == r["hbm"]["achieved"]
    assert len(r["per_stage"]) == 4 and r["bytes_per_cell_step"] == 768 and 0.5 < r["stage_kernel_share_of_step"] <= 1.05
    assert len(r["library_build_id"]) == 12
    # nothing typed in: the ncu side of the roofline is there only when a committed capture of this workload exists
    assert (r["traffic"] is None) == (r["traffic_source"] is None) == (r["alu"] is None)
    assert d["repeats"]["n"] == 3 and len(d["repeats"]["ms_per_step"]) == 3
    assert d["repeats"]["best_ms_per_step"] <= d["ms_per_step"] <= max(d["repeats"]["ms_per_step"])
    e = d["e2e"]
    nbytes = 64 * d["config"]["nz"] * d["config"]["nv"]
    assert e["h2d_bytes_per_step"] == nbytes and e["d2h_bytes_per_step"] == nbytes and 0 < e["value"] < d["value"]
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(d["clocks"])
    assert d["graph_replay"]["value"] > 0
    c = d["checks"]
    assert c["steps_total"] == 3 + 3 * 20 + 20                   # warm-up, 3 timed repeats, event-free (graph) pass
    if workload != "cfg1":      # z-homogeneous start without the vacuum term: trace per cell and M0 stay put
        assert c["trace_dev_max"] < 1e-12 and c["dM0_max"] < 1e-8
    else:                       # omega != 0: only the projection of M0 on B is conserved (reading R2)
        assert abs(c["B_dot_dM0"]) < 1e-8 * max(1.0, c["M0_scale"])
    if decomp == "slab":
        assert "z-slabs x1" in d["config"]["parallelism"]
    assert d["secondary"] == []


def test_bench_secondary_lines():
    """The default line carries the other kernel families: cfg3 (FD4+KO3, own roofline and clocks) and the launch-bound grids."""
    d = _run("--workload", "cfg2", "--steps", "20")
    names = [x["workload"] for x in d["secondary"]]
    assert names == ["cfg3", "cfg0", "cfg1", "cfg2"]
    s3 = d["secondary"][0]
    assert s3["roofline"]["bound"] == "hbm" and s3["roofline"]["frac"] > 0.5 and s3["clocks"]["sm_mhz"] > 0
    assert s3["config"]["scheme"] == "FD4_KO3" and s3["value"] > 1e9
    for x in d["secondary"][1:]:
        assert 0 < x["graph_replay"]["ms_per_step"] <= 1.5 * x["launch_by_launch"]["ms_per_step"]


def test_slab_bitwise_check_of_the_multi_gpu_line():
    """bench.py's N > 1 line carries `slab_check` (a reduced free-running slab run against the single domain, bit for bit);
    with one rank the slab is linked to itself."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    sys.path.insert(0, ROOT)
    import bench
    r = bench.slab_bitwise_check(1, 0)
    assert r["bitwise_equal_to_single_domain"] is True and r["halo_wait_failed"] is False and r["slabs"] == 1
