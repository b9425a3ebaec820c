#!/usr/bin/env python
"""bench.py -- throughput of the COSEnu RK4 hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl ours|reference]

A "step" is one classical RK4 step (4 fused stage launches) of the whole (z,v) grid.  metric =
(z,v) cell-updates per second per RK4 step, fp64.  Default workload: BASELINE.json configs[4]
(WENO7, 262144 x 512), the largest single-GPU configuration, on which the north-star target is quoted;
`--workload cfg3` is the bandwidth-scale FD4+KO3 run.  Inputs are seeded and synthetic
(paper_2203_12866_b200/inputs.py); the state (>= 2 GB per copy) is far larger than L2, so no L2 flush
is needed between steps.

N > 1 (torchrun): by default every rank owns an independent replica of the workload on its own GPU (weak
scaling, no data-path collective; the north star is a one-GPU path).  `--decomp slab` runs ONE periodic grid
of N x nz rows cut into z-slabs, one per rank: the halo exchange is fused into the stage kernels (peer stores
over NVLink + arrival counters); still weak scaling (nz rows per GPU).  Barrier +
max-over-ranks timing; value = total cells of all ranks / that time.  With N = 1, `--decomp slab` runs the
slab code path on a slab linked to itself.

--impl reference: the CPU oracle (oracle/, as it stands) timed on the host cores on a bounded sample of
the same workload (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "(z,v) cell-updates/sec per RK4 step (fp64)"
UNIT = "cell-updates/s"
# algorithmic HBM bytes per cell per stage launch:
# read stage input + u0 + acc, write stage output + acc, 64 B each
# per RK formulation (cosenu.h COSENU_OPT_RK_FORM): bytes per cell of stages 1..4
STAGE_BYTES = {0: [192, 320, 320, 192], 1: [128, 256, 320, 192], 2: [128, 192, 192, 320], 3: [128, 256, 192, 192]}
STAGE_KERNEL = {0: ["FIRST", "MID", "MID", "LAST"], 1: ["FIRST_LEAN", "MID_REBUILD", "MID", "LAST"],
                2: ["FIRST_LEAN", "MID_NOACC", "MID_NOACC", "LAST_COMB"],
                3: ["FIRST_LEAN", "MID_P", "MID_NOACC", "LAST_P"]}
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant stage launch from the
# committed ncu capture (profiles/r01_traffic_*.csv), per (workload, rk_form); None where not captured
NCU_TRAFFIC_BYTES = {("cfg4", 2): 44279386880, ("cfg3", 2): 10752631296,   # profiles/r01_traffic_*.csv, RK stage 4 (LAST_COMB)
                     ("cfg4", 3): 34396154624, ("cfg3", 3): 8674394880}    # profiles/r01b_traffic_*.csv, RK stage 2 (MID_P)


# fp64 instructions (DFMA + DMUL + DADD, per thread = per (z,v) cell) one stage launch executes per cell, from
# smsp__sass_thread_inst_executed_op_d{fma,mul,add}_pred_on.sum of the committed capture (profiles/r01b_fp64_*.csv): the
# ALU side of the roofline.  Peak = 148 SMs x 4 sub-partitions x 16 fp64 lanes per clock x 1.965 GHz.
FP64_PER_CELL = {"WENO7": {"FIRST_LEAN": 618.3, "MID_P": 647.2, "MID_NOACC": 620.5, "LAST_P": 626.3},
                 "FD4_KO3": {"FIRST_LEAN": 151.9, "MID_P": 175.9, "MID_NOACC": 151.9, "LAST_P": 159.9}}
FP64_PEAK_LANE_OPS = 148 * 4 * 16 * 1.965e9


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.p = index, None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
            out, _ = self.p.communicate()
        sm, mx, reasons, pw = [], [], set(), []
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(x, device="cuda"):
    """Max of a per-rank scalar over all ranks (the job is as slow as its slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cells, steps, world, ms):
    """Whole-job aggregate: every rank advances its own `cells` grid by `steps` steps (weak scaling)."""
    return world * cells * steps / (ms * 1e-3)


def workload(name):
    from paper_2203_12866_b200 import inputs
    c = dict(inputs.CONFIGS[name])
    c["name"] = name
    return c


def oracle_sample(c, target_s=15.0, max_nz=4096):
    """Time the oracle, as it stands, on a z-reduced sample of workload c (same nv, scheme, physics)."""
    from oracle import cosenu_ref as R
    from paper_2203_12866_b200 import inputs
    nz = min(c["nz"], max_nz)
    cores = os.cpu_count() or 1
    st = inputs.config_state(c["name"], nz=nz)
    r = R.RefSim(nz, c["nv"], float(nz) * (c["L"] / c["nz"]), c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"])
    r.set_state(st)
    t0 = time.perf_counter(); r.step(1); t1 = time.perf_counter() - t0      # also the warm-up
    n = int(max(1, min(200, target_s / max(t1, 1e-3))))
    t0 = time.perf_counter(); r.step(n); dt = time.perf_counter() - t0
    # the same oracle on ONE thread ("timed at 1 thread and at all cores"), a few steps only
    r.set_option(R.OPT_THREADS, 1)
    n1 = int(max(1, min(n, 4.0 / max(t1 * cores, 1e-3))))
    t0 = time.perf_counter(); r.step(n1); dt1 = time.perf_counter() - t0
    r.close()
    return {"value": nz * c["nv"] * n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "value_1_thread": nz * c["nv"] * n1 / dt1,
            "sample": "%s with nz reduced to %d (nv=%d), %d RK4 steps, OpenMP over z on %d threads, %.1f s (+ %d steps on 1 thread, %.1f s)"
                      % (c["name"], nz, c["nv"], n, cores, dt, n1, dt1)}, nz, n, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = workload(args.workload)
    from oracle import cosenu_ref as R
    from paper_2203_12866_b200 import inputs
    nz = min(c["nz"], 2048)
    st = inputs.config_state(c["name"], nz=nz)
    r = R.RefSim(nz, c["nv"], float(nz) * (c["L"] / c["nz"]), c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"])
    r.set_state(st)
    for _ in range(args.warmup):
        r.step(1)
    t0 = time.perf_counter()
    r.step(args.steps)
    dt = time.perf_counter() - t0
    r.close()
    cores = os.cpu_count() or 1
    val = nz * c["nv"] * args.steps / dt
    sample = "%s with nz reduced to %d (nv=%d): each step = one RK4 step of that sample; OpenMP over z, %d threads" % (
        c["name"], nz, c["nv"], cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": c["name"], "scheme": "FV_WENO7" if c["scheme"] else "FD4_KO3", "nz": c["nz"],
                   "nv": c["nv"], "sample_nz": nz},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2203_12866_b200 import binding as B
    from paper_2203_12866_b200 import inputs

    c = workload(args.workload)
    nz, nv = c["nz"], c["nv"]
    cells = nz * nv
    # ---- synthetic seeded input, built on the host in pinned memory (the e2e leg copies from it)
    host = torch.empty((8, nz, nv), dtype=torch.float64, pin_memory=True)
    hnp = host.numpy()
    if args.decomp != "slab":
        hnp[...] = inputs.fast_conversion_state(nz, nv, c["seed"] + rank) if c["kind"] == "fast" else \
            inputs.vacuum_check_state(nz, nv, c["seed"] + rank)
    if args.decomp == "slab":
        # one periodic grid of world * nz rows, this rank's slab of nz rows; the library builds the slab's rows of the
        # seeded global state (cosenu_init enters the splitmix64 stream at z_begin)
        if c["kind"] != "fast":
            raise SystemExit("bench.py --decomp slab: fast-conversion workloads only")
        from paper_2203_12866_b200 import slab as S
        sim = S.CosenuSlab(world * nz, nv, world * c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"],
                           rk_form=args.rk_form, variant=args.variant)
        sim.init(c["seed"])
        sim.get_state(host)
        api = sim.sim
    else:
        sim = B.Cosenu(nz, nv, c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"], rk_form=args.rk_form,
                       variant=args.variant)
        sim.set_state(host)
        api = sim
    d0 = sim.diagnostics()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps
    sim.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    api.set_option(B.OPT_STAGE_TIMING, 1)       # CUDA events around every stage launch, on the launching stream
    l0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    sim.step(args.steps)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count() - l0
    stage_ms, nst = api.stage_times()
    api.set_option(B.OPT_STAGE_TIMING, 0)
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(ms)
    value = whole_job_value(cells, args.steps, world, ms)

    # ---- the same K steps without the per-stage events: cosenu_step replays its CUDA graph (8 steps per launch) when
    # it may (single domain).  Matters on the small, launch-bound grids only; reported beside `value`.
    barrier()
    e0.record()
    sim.step(args.steps)
    e1.record()
    barrier()
    ms_graph = max_over_ranks(e0.elapsed_time(e1))
    graph_replay = {"value": whole_job_value(cells, args.steps, world, ms_graph), "unit": UNIT,
                    "ms_per_step": ms_graph / args.steps,
                    "what": "same K steps, no per-stage events; CUDA-graph replay when steps >= 16 and single domain"}

    # ---- invariants at the bench size (properties that hold at any size)
    d1 = sim.diagnostics()
    checks = {"steps_total": d1["step"], "dM0_max": max(abs(x) for x in d1["dM0"]),
              "psurv_nu": d1["psurv_nu"], "trace_dev_max": d1["trace_dev_max"], "dP_max": d1["dP_max"]}

    # ---- end to end through the public API with HOST buffers: H2D of the state, one RK4 step, D2H of the result
    ne2e = max(1, args.e2e_steps)
    sim.set_state(host); sim.step(1); sim.get_state(host)     # warm-up of the e2e path
    barrier()
    t0 = time.perf_counter()
    for _ in range(ne2e):
        sim.set_state(host)
        sim.step(1)
        sim.get_state(host)       # synchronises
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s)
    state_bytes = 8 * cells * 8
    e2e = {"value": world * cells * ne2e / e2e_s, "unit": UNIT, "h2d_bytes_per_step": state_bytes,
           "d2h_bytes_per_step": state_bytes, "steps": ne2e,
           "what": "cosenu_set_state(pinned host) + cosenu_step(1) + cosenu_get_state(pinned host) per step"}
    sim.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel = the stage launch with the longest average duration
    peak, peak_src = measured_peaks()
    sb = STAGE_BYTES[args.rk_form]
    step_bytes = sum(sb)
    avg = [stage_ms[k] / max(nst, 1) for k in range(4)]
    per_stage = [{"stage": k + 1, "kernel": STAGE_KERNEL[args.rk_form][k], "bytes_per_cell": sb[k], "avg_ms": avg[k],
                  "GBps": sb[k] * cells / (avg[k] * 1e-3) / 1e9} for k in range(4)] if nst else []
    dom = max(range(4), key=lambda k: avg[k]) if nst else 0
    achieved = per_stage[dom]["GBps"] if nst else None
    # the same launch against the plain fp64 ALU peak (WENO7 is co-bound by it; FD is not)
    sname = "WENO7" if c["scheme"] else "FD4_KO3"
    nfp = FP64_PER_CELL[sname].get(STAGE_KERNEL[args.rk_form][dom]) if nst else None
    alu = None
    if nfp:
        a = nfp * cells / (avg[dom] * 1e-3)
        alu = {"achieved": a / 1e12, "peak": FP64_PEAK_LANE_OPS / 1e12, "unit": "T fp64 instr/s (per lane; x2 for FMA flops)",
               "frac": a / FP64_PEAK_LANE_OPS, "fp64_instr_per_cell_launch": nfp,
               "peak_source": "148 SMs x 4 SMSPs x 16 lanes/clk x 1.965 GHz (max SM clock; sustained clock is lower under sw_power_cap)"}
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak if achieved else None,
                "traffic": NCU_TRAFFIC_BYTES.get((c["name"], args.rk_form)), "peak_source": peak_src,
                "kernel": "stage_kernel<%s, %s> (RK stage %d)" % ("WENO7" if c["scheme"] else "FD4_KO3",
                                                                  STAGE_KERNEL[args.rk_form][dom], dom + 1),
                "algorithmic_bytes_per_launch": sb[dom] * cells, "avg_launch_ms": avg[dom],
                "stage_kernel_share_of_step": sum(avg) / (ms / args.steps) if nst else None,
                "alu": alu, "per_stage": per_stage, "bytes_per_cell_step": step_bytes,
                "step_model_GBps": step_bytes * value / world / 1e9,
                "step_model_frac": step_bytes * value / world / 1e9 / peak,
                # "effective" bandwidth with the fused 3-array traffic model (1024 B per cell-step),
                # whatever carrier the run used; 70 % of the measured peak with this model = 4.47 G cell-updates/s
                "survey_model_1024B": {"GBps": 1024 * value / world / 1e9, "frac_of_measured_peak": 1024 * value / world / 1e9 / peak,
                                       "frac_of_8TBps_nominal": 1024 * value / world / 1e9 / 8000.0}}
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu, _, _, _ = oracle_sample(c)
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": c["name"], "scheme": "FV_WENO7" if c["scheme"] else "FD4_KO3", "nz": nz, "nv": nv,
                      "dt": c["dt"], "omega": c["omega"], "theta": c["theta"], "mu": c["mu"],
                      "state_bytes_per_copy": state_bytes, "l2": "inputs larger than L2 (no flush needed)",
                      "parallelism": ("z-slabs x%d of one grid of %d rows (halo exchange fused into the stage kernels)"
                                      % (world, world * nz)) if args.decomp == "slab" else "replicas x%d" % world,
                      "rk_form": args.rk_form, "variant": args.variant},
           "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
           "graph_replay": graph_replay, "checks": checks}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg4", choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--rk-form", type=int, default=3, choices=[0, 1, 2, 3])
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"])
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
