#!/usr/bin/env python
"""bench.py -- throughput of the COSEnu RK4 hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl ours|reference]

A "step" is one classical RK4 step (4 fused stage launches) of the whole (z,v) grid.  metric =
(z,v) cell-updates per second per RK4 step, fp64.  Default workload: BASELINE.json configs[4]
(WENO7, 262144 x 512), the largest single-GPU configuration, on which the north-star target is quoted.
Inputs are seeded and synthetic (paper_2203_12866_b200/inputs.py); the state (>= 2 GB per copy) is far larger than
L2, so no L2 flush is needed between steps.  The timed region of K steps is repeated 3 times: `value` is the median,
the best is in `repeats`.  The same line carries `secondary`: the bandwidth-scale FD4+KO3 run (cfg3, with its own
roofline and clocks) and the launch-bound grids cfg0-cfg2 (ms per step launch by launch and as CUDA-graph replays).
`roofline` leads with what binds the dominant launch ("alu": the plain fp64 pipe, WENO7; "hbm": FD4+KO3); the per-stage
ncu counters it quotes (DRAM bytes, fp64 instructions) are read from the committed capture profiles/r03_metrics_*.csv.

N > 1 (torchrun): ONE periodic grid of N x nz rows cut into z-slabs, one per rank: the halo exchange is fused into
the stage kernels (peer stores over NVLink + arrival counters); weak scaling (nz rows per
GPU), free-running ranks.  Beside it: N independent replicas (`other_decomposition`) and a bitwise check of a reduced
slab run against the single domain (`slab_check`).  A halo wait that timed out invalidates the slab figure: the line
then reports the replicas and the flag.  `--decomp replicas|slab` forces one of them (N = 1 with slab: a slab linked
to itself).  Barrier + max-over-ranks timing; value = total cells of all ranks / that time.

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
# plain fp64 ALU peak: 148 SMs x 4 sub-partitions x 16 fp64 lanes per clock (one DFMA/DMUL/DADD warp instruction per 2 clk
# and sub-partition, measured: DESIGN.md section 5) x the SM clock
FP64_LANES_PER_CLK = 148 * 4 * 16
SM_MAX_MHZ = 1965.0
REPEATS = 3          # repeats of the timed region (best and median of >= 3)
PROFILE_ROUND = "r03"


def library_build_id():
    """The id compiled into the library that is actually loaded (cosenu_build_id: sha1 over the sources it was built from),
    so that a stale prebuilt .so cannot carry a fresh id."""
    from paper_2203_12866_b200 import binding
    return binding.build_id()


def source_build_id():
    """The same hash over the sources as they sit in the tree right now."""
    from paper_2203_12866_b200 import build
    return build.source_id()


def profile_build_id():
    """The library build id the committed ncu capture of this round was taken on (stated in the .md beside the .csv files)."""
    import re
    path = os.path.join(ROOT, "profiles", "%s_launches.md" % PROFILE_ROUND)
    if not os.path.exists(path):
        return None
    m = re.search(r"[Ll]ibrary build id[^`]*`([0-9a-f]{12})`", open(path).read())
    return m.group(1) if m else None


def load_profile(workload, rk_form, variant):
    """Per-stage ncu counters of the committed capture profiles/<round>_metrics_<workload>.csv (one RK4 step = 4 launches,
    in launch order; the command that wrote it is in the .md beside it): DRAM bytes, fp64 thread instructions, FP64-pipe
    activity.  None when there is no capture of this workload / RK carrier / kernel shape: nothing is typed into this file."""
    import csv
    if rk_form != 3 or variant not in (0, 4):
        return None
    path = os.path.join(ROOT, "profiles", "%s_metrics_%s.csv" % (PROFILE_ROUND, workload))
    if not os.path.exists(path):
        return None
    if profile_build_id() != library_build_id():
        return None     # a capture of another binary is not quoted (roofline.traffic_source says so)
    per = {}
    with open(path) as f:
        rows = list(csv.reader(f))
    hdr = next((r for r in rows if "Metric Name" in r and "Kernel Name" in r), None)
    if hdr is None:
        return None
    ci, ck, cm, cv = hdr.index("ID"), hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value")
    for r in rows:
        if len(r) != len(hdr) or not r[ci].isdigit():
            continue
        d = per.setdefault(int(r[ci]), {"kernel": r[ck]})
        try:
            d[r[cm]] = float(r[cv].replace(",", ""))
        except ValueError:
            pass
    ids = sorted(per)
    if len(ids) < 4:
        return None
    out = []
    for k in ids[:4]:
        d = per[k]
        fp = sum(d.get("smsp__sass_thread_inst_executed_op_%s_pred_on.sum" % o, 0.0) for o in ("dadd", "dfma", "dmul"))
        out.append({"kernel": d["kernel"].split("(")[0].replace("void ", ""),
                    "dram_bytes": d.get("dram__bytes_read.sum", 0.0) + d.get("dram__bytes_write.sum", 0.0),
                    "fp64_thread_inst": fp,
                    "fp64_pipe_pct": d.get("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
                    "ncu_ms": d.get("gpu__time_duration.sum", 0.0) * 1e-6})
    return {"file": os.path.relpath(path, ROOT), "stages": out}


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


def make_state(c, nz, nv, rank, pinned=True):
    """Seeded synthetic input of workload c in pinned host memory (the e2e leg copies from it)."""
    import torch
    from paper_2203_12866_b200 import inputs
    host = torch.empty((8, nz, nv), dtype=torch.float64, pin_memory=pinned)
    host.numpy()[...] = inputs.fast_conversion_state(nz, nv, c["seed"] + rank) if c["kind"] == "fast" else \
        inputs.vacuum_check_state(nz, nv, c["seed"] + rank)
    return host


def timed_steps(sim, api, B, steps, barrier, repeats=REPEATS):
    """`repeats` timed regions of exactly `steps` RK4 steps each, CUDA events on the launching stream around the region and
    around every stage launch inside it (COSENU_OPT_STAGE_TIMING).  Returns the per-repeat ms (max over ranks) and the
    per-stage sums."""
    import torch
    api.set_option(B.OPT_STAGE_TIMING, 1)
    ms_all, launches = [], 0
    stage_sum, nst = [0.0] * 4, 0
    for _ in range(repeats):
        l0 = sim.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        sim.step(steps)
        e1.record()
        barrier()
        ms_all.append(max_over_ranks(e0.elapsed_time(e1)))
        launches = sim.launch_count() - l0
        sm, n = api.stage_times()
        stage_sum = [a + b for a, b in zip(stage_sum, sm)]
        nst += n
    api.set_option(B.OPT_STAGE_TIMING, 0)
    return ms_all, launches, stage_sum, nst


def median(x):
    y = sorted(x)
    return y[len(y) // 2] if len(y) % 2 else 0.5 * (y[len(y) // 2 - 1] + y[len(y) // 2])


def roofline_block(c, rk_form, variant, cells, avg, step_ms, value_per_gpu, clocks):
    """Roofline of the dominant kernel = the stage launch with the longest mean duration, against what binds it: the HBM
    copy peak (FD4+KO3) or the plain fp64 ALU peak (WENO7); the other side is reported next to it."""
    peak, peak_src = measured_peaks()
    sb = STAGE_BYTES[rk_form]
    names = STAGE_KERNEL[rk_form]
    sname = "WENO7" if c["scheme"] else "FD4_KO3"
    prof = load_profile(c["name"], rk_form, variant)
    per_stage = []
    for k in range(4):
        d = {"stage": k + 1, "kernel": names[k], "bytes_per_cell": sb[k], "avg_ms": avg[k],
             "GBps": sb[k] * cells / (avg[k] * 1e-3) / 1e9}
        if prof:
            ps = prof["stages"][k]
            d["fp64_instr_per_cell"] = ps["fp64_thread_inst"] / cells
            d["T_fp64_instr_per_s"] = ps["fp64_thread_inst"] / (avg[k] * 1e-3) / 1e12
            d["ncu_dram_bytes"] = ps["dram_bytes"]
            d["ncu_fp64_pipe_pct"] = ps["fp64_pipe_pct"]
        per_stage.append(d)
    dom = max(range(4), key=lambda k: avg[k])
    hbm = {"achieved": per_stage[dom]["GBps"], "peak": peak, "unit": "GB/s", "frac": per_stage[dom]["GBps"] / peak,
           "algorithmic_bytes_per_launch": sb[dom] * cells, "peak_source": peak_src}
    sm_mhz = (clocks or {}).get("sm_mhz") or SM_MAX_MHZ
    alu = None
    if prof:
        a = per_stage[dom]["T_fp64_instr_per_s"]
        pk = FP64_LANES_PER_CLK * SM_MAX_MHZ * 1e6 / 1e12
        pk_s = FP64_LANES_PER_CLK * sm_mhz * 1e6 / 1e12
        alu = {"achieved": a, "peak": pk, "unit": "T fp64 instr/s (DFMA + DMUL + DADD per lane; an FMA counts once)",
               "frac": a / pk, "peak_at_sampled_clock": pk_s, "frac_at_sampled_clock": a / pk_s, "sampled_sm_mhz": sm_mhz,
               "fp64_instr_per_cell_launch": per_stage[dom]["fp64_instr_per_cell"],
               "peak_source": "148 SMs x 4 sub-partitions x 16 fp64 lanes/clk x SM clock (DESIGN.md section 5): at the maximum "
                              "clock %.0f MHz and at the clock sampled during the timed region" % SM_MAX_MHZ}
    bound = "alu" if (sname == "WENO7" and alu is not None and alu["frac_at_sampled_clock"] >= hbm["frac"]) else "hbm"
    lead = alu if bound == "alu" else hbm
    r = {"bound": bound, "achieved": lead["achieved"], "peak": lead["peak"], "unit": lead["unit"], "frac": lead["frac"],
         "traffic": per_stage[dom].get("ncu_dram_bytes"),
         "traffic_source": (prof["file"] + " (committed ncu capture of `bench.py --workload %s --steps 2 --warmup 5 --no-cpu-baseline "
                            "--no-secondary --e2e-steps 1` on the same library build, not measured in this run; full command in "
                            "profiles/%s_launches.md)" % (c["name"], PROFILE_ROUND)) if prof else None,
         # a committed capture of this workload exists but names another binary: it is not quoted, and this says why
         "traffic_not_quoted": ("profiles/%s_launches.md was captured on library build %s, the loaded library is %s"
                                % (PROFILE_ROUND, profile_build_id(), library_build_id()))
         if (prof is None and rk_form == 3 and variant in (0, 4) and profile_build_id() != library_build_id()
             and os.path.exists(os.path.join(ROOT, "profiles", "%s_metrics_%s.csv" % (PROFILE_ROUND, c["name"])))) else None,
         "kernel": "%s (RK stage %d, %s)" % (prof["stages"][dom]["kernel"] if prof else "stage kernel", dom + 1, names[dom]),
         "avg_launch_ms": avg[dom], "stage_kernel_share_of_step": sum(avg) / step_ms,
         "hbm": hbm, "alu": alu, "per_stage": per_stage, "bytes_per_cell_step": sum(sb),
         "step_GBps": sum(sb) * value_per_gpu / 1e9, "step_frac_of_hbm_peak": sum(sb) * value_per_gpu / 1e9 / peak,
         "library_build_id": library_build_id(), "library_matches_sources": library_build_id() == source_build_id()}
    return r


def invariants(c, d1):
    """Properties that hold at any size: with omega != 0 only the projection of M0 on
    B = (sin 2 theta, 0, -cos 2 theta) is conserved (reading R2), otherwise all of M0."""
    import math
    out = {"steps_total": d1["step"], "psurv_nu": d1["psurv_nu"], "trace_dev_max": d1["trace_dev_max"], "dP_max": d1["dP_max"]}
    if c["omega"] != 0.0:
        bx, bz = math.sin(2 * c["theta"]), -math.cos(2 * c["theta"])
        out["B_dot_dM0"] = bx * d1["dM0"][0] + bz * d1["dM0"][2]
        out["M0_scale"] = max(abs(x) for x in d1["M0"])
    else:
        out["dM0_max"] = max(abs(x) for x in d1["dM0"])
    return out


def bench_workload(args, name, steps, warmup, world, rank, local, decomp, e2e_steps, sample_clocks):
    """One workload, device-resident + (optionally) end to end.  Returns the result dict of rank 0 (None on other ranks)."""
    import torch
    import torch.distributed as dist
    from paper_2203_12866_b200 import binding as B
    c = workload(name)
    nz, nv = c["nz"], c["nv"]
    cells = nz * nv

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    host = make_state(c, nz, nv, rank) if decomp != "slab" else torch.empty((8, nz, nv), dtype=torch.float64, pin_memory=True)
    if decomp == "slab":
        # one periodic grid of world * nz rows, this rank's slab of nz rows; the library builds the slab's rows of the
        # seeded global state (cosenu_init enters the splitmix64 stream at z_begin)
        if c["kind"] != "fast":
            raise SystemExit("bench.py --decomp slab: fast-conversion workloads only")
        from paper_2203_12866_b200 import slab as S
        sim = S.CosenuSlab(world * nz, nv, world * c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"],
                           rk_form=args.rk_form, variant=args.variant)
        api = sim.sim
        # ranks reach their first step at different times (uploads, the e2e leg's 8.6 GB copies): a halo wait that gives up
        # after the default 4 s would turn one slow rank into "halo_wait_failed"
        api.set_option(B.OPT_HALO_TIMEOUT_S, 60.0)
        sim.init(c["seed"])
        sim.get_state(host)
    else:
        sim = B.Cosenu(nz, nv, c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"], rk_form=args.rk_form,
                       variant=args.variant)
        sim.set_state(host)
        api = sim

    # ---- device-resident throughput: W warm-up steps, then REPEATS timed regions of exactly K steps
    barrier()            # every rank holds its state (and, decomposed, its neighbours' ghost rows) before anybody steps
    sim.step(warmup)
    barrier()
    sampler = ClockSampler(local) if (sample_clocks and rank == 0) else None
    if sampler:
        sampler.start()
        time.sleep(0.15)
    ms_all, launches, stage_sum, nst = timed_steps(sim, api, B, steps, barrier)
    clocks = sampler.stop() if sampler else None
    ms = median(ms_all)
    value = whole_job_value(cells, steps, world, ms)

    # ---- the same K steps without the per-stage events: cosenu_step replays its CUDA graph (8 steps per launch) when
    # it may (single domain).  Matters on the small, launch-bound grids only; reported beside `value`.
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    sim.step(steps)
    e1.record()
    barrier()
    ms_graph = max_over_ranks(e0.elapsed_time(e1))

    halo_failed = False
    if decomp == "slab":
        halo_failed = bool(max_over_ranks(1.0 if sim.wait_failed() else 0.0))
    d1 = sim.diagnostics()

    # ---- end to end through the public API with HOST buffers: H2D of the state, one RK4 step, D2H of the result
    e2e = None
    if e2e_steps > 0:
        sim.set_state(host); sim.step(1); sim.get_state(host)     # warm-up of the e2e path
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            sim.set_state(host)
            sim.step(1)
            sim.get_state(host)       # synchronises
        barrier()
        e2e_s = max_over_ranks(time.perf_counter() - t0)
        state_bytes = 8 * cells * 8
        e2e = {"value": world * cells * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": state_bytes,
               "d2h_bytes_per_step": state_bytes, "steps": e2e_steps,
               "what": "cosenu_set_state(pinned host) + cosenu_step(1) + cosenu_get_state(pinned host) per step"}
    sim.close()
    del host
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    avg = [stage_sum[k] / max(nst, 1) for k in range(4)]
    return {"workload": name, "c": c, "cells": cells, "value": value, "ms_per_step": ms / steps,
            "repeats": {"n": len(ms_all), "ms_per_step": [m / steps for m in ms_all], "best_ms_per_step": min(ms_all) / steps,
                        "median_ms_per_step": ms / steps, "best_value": whole_job_value(cells, steps, world, min(ms_all))},
            "graph_replay": {"value": whole_job_value(cells, steps, world, ms_graph), "unit": UNIT, "ms_per_step": ms_graph / steps,
                             "what": "same K steps, no per-stage events; CUDA-graph replay when steps >= 16 and single domain"},
            "clocks": clocks, "launches": launches, "e2e": e2e, "checks": invariants(c, d1), "halo_wait_failed": halo_failed,
            "roofline": roofline_block(c, args.rk_form, args.variant, cells, avg, ms / steps, value / world, clocks)}


def config_of(r, args, world, decomp):
    c = r["c"]
    return {"workload": c["name"], "scheme": "FV_WENO7" if c["scheme"] else "FD4_KO3", "nz": c["nz"], "nv": c["nv"],
            "dt": c["dt"], "omega": c["omega"], "theta": c["theta"], "mu": c["mu"],
            "state_bytes_per_copy": 8 * r["cells"] * 8, "l2": "inputs larger than L2 (no flush needed)" if r["cells"] * 64 > 4 * 126e6
            else "state of %.1f MB fits in L2: launch-bound grid, reported in `secondary` only" % (r["cells"] * 64 / 1e6),
            "parallelism": ("z-slabs x%d of one grid of %d rows (halo exchange fused into the stage kernels: the data plane is "
                            "peer-memory stores + arrival counters over NVLink, NOT NCCL; torch.distributed/NCCL carries only the "
                            "set-up descriptors, the diagnostics' few sums and the barriers)"
                            % (world, world * c["nz"])) if decomp == "slab" else "replicas x%d" % world,
            "rk_form": args.rk_form, "variant": args.variant}


def small_grid(args, name):
    """Launch-bound grids (configs 0-2): ms per step launch by launch and as CUDA-graph replays, one GPU."""
    import torch
    from paper_2203_12866_b200 import binding as B
    c = workload(name)
    nz, nv = c["nz"], c["nv"]
    host = make_state(c, nz, nv, 0, pinned=False)
    out = {"workload": name, "scheme": "FV_WENO7" if c["scheme"] else "FD4_KO3", "nz": nz, "nv": nv}
    steps = 400 if nz * nv < (1 << 22) else 64
    for key, graph in (("launch_by_launch", False), ("graph_replay", True)):
        sim = B.Cosenu(nz, nv, c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"], rk_form=args.rk_form,
                       variant=args.variant, graph=graph)
        sim.set_state(host)
        sim.step(32)
        torch.cuda.synchronize()
        ms = []
        for _ in range(REPEATS):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); sim.step(steps); e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1) / steps)
        sim.close()
        out[key] = {"ms_per_step": median(ms), "best_ms_per_step": min(ms), "value": nz * nv / (median(ms) * 1e-3), "unit": UNIT}
    return out


def slab_bitwise_check(world, rank, scheme=1):
    """A reduced grid cut into one z-slab per rank, free-running (no host synchronisation between the stages), against the
    single-domain run of the same grid on rank 0: bit for bit.  Collective."""
    import numpy as np
    import torch.distributed as dist
    from paper_2203_12866_b200 import binding as B
    from paper_2203_12866_b200 import slab as S
    nzl, nv, nsteps = 148 * 16, 64, 12
    nz = world * nzl
    args = (nz, nv, float(nz), 0.4, 1e-2, 0.01, 1.0, scheme)
    sl = S.CosenuSlab(*args)
    sl.init(4242)
    sl.step(nsteps)
    failed = False
    try:
        sl.sync()
        mine = sl.get_state()
    except B.CosenuError:
        failed, mine = True, np.zeros((8, sl.nz, nv))
    parts = [None] * world if rank == 0 else None
    if world > 1:
        dist.gather_object(mine, parts, dst=0)
    else:
        parts = [mine]
    sl.close()
    ok = None
    if rank == 0:
        ref = B.Cosenu(*args)
        ref.init(4242)
        ref.step(nsteps)
        ok = (not failed) and bool(np.array_equal(np.concatenate(parts, axis=1), ref.get_state()))
        ref.close()
    return {"nz": nz, "nv": nv, "steps": nsteps, "slabs": world, "bitwise_equal_to_single_domain": ok, "halo_wait_failed": failed}


def run_ours(args):
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
    c = workload(args.workload)

    # N = 1: the single domain (--decomp slab: the slab code path on a slab linked to itself).
    # N > 1: ONE periodic grid of N x nz rows cut into z-slabs, one per rank, halo exchange fused into the stage kernels (the
    # multi-GPU design of this repo; weak scaling) -- and, beside it, N independent replicas.  `value` is
    # the slab figure unless a halo wait failed (then the run is invalid and the replica figure is reported, with the flag).
    decomp = args.decomp or ("slab" if world > 1 else "replicas")
    main_r = bench_workload(args, args.workload, args.steps, args.warmup, world, rank, local, decomp, max(1, args.e2e_steps), True)
    other, check = None, None
    if world > 1 and not args.decomp:
        other = bench_workload(args, args.workload, args.steps, args.warmup, world, rank, local, "replicas", 0, False)
        check = slab_bitwise_check(world, rank)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    exit_code = 0
    if main_r["halo_wait_failed"]:
        # stale ghost rows: the throughput of a corrupted run is not a result
        exit_code = 3
        if other is not None:
            main_r, other, decomp = other, main_r, "replicas"
            exit_code = 0
    secondary = []
    if world == 1 and not args.no_secondary:
        if args.workload != "cfg3":   # the HBM-bound kernel family at bandwidth scale
            r = bench_workload(args, "cfg3", max(args.steps, 20), args.warmup, 1, 0, local, "replicas", 0, True)
            secondary.append({"workload": "cfg3", "config": config_of(r, args, 1, "replicas"), "value": r["value"], "unit": UNIT,
                              "ms_per_step": r["ms_per_step"], "repeats": r["repeats"], "clocks": r["clocks"],
                              "roofline": r["roofline"], "checks": r["checks"]})
        for name in ("cfg0", "cfg1", "cfg2"):
            secondary.append(small_grid(args, name))
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu, _, _, _ = oracle_sample(c)
    out = {"metric": METRIC, "value": main_r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": main_r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": config_of(main_r, args, world, decomp),
           "timing": "median of %d repeats of the timed region of K steps; the per-stage CUDA events (COSENU_OPT_STAGE_TIMING, five event "
                     "records per step on the launching stream, launch by launch, no CUDA-graph replay) are ON inside it; the first "
                     "repeat is usually the fastest (the board's power controller), all are in `repeats`; `graph_replay` is the same "
                     "workload replayed from a CUDA graph without events" % REPEATS, "repeats": main_r["repeats"],
           "clocks": main_r["clocks"], "e2e": main_r["e2e"], "gpu_launches": main_r["launches"], "roofline": main_r["roofline"],
           "cpu_baseline": cpu, "graph_replay": main_r["graph_replay"], "checks": main_r["checks"], "secondary": secondary}
    if world > 1:
        out["halo_wait_failed"] = bool(main_r["halo_wait_failed"] or (other or {}).get("halo_wait_failed", False))
        if other is not None:
            out["other_decomposition"] = {"parallelism": "replicas x%d" % world if decomp == "slab" else "z-slabs x%d" % world,
                                          "value": other["value"], "unit": UNIT, "ms_per_step": other["ms_per_step"],
                                          "halo_wait_failed": other["halo_wait_failed"]}
        out["slab_check"] = check
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    if exit_code:
        sys.exit(exit_code)


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
    ap.add_argument("--no-secondary", action="store_true", help="skip the `secondary` lines (cfg3 and the launch-bound grids)")
    ap.add_argument("--decomp", default=None, choices=["replicas", "slab"],
                    help="default: single domain at N = 1; at N > 1 one grid cut into z-slabs, with N replicas beside it")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
