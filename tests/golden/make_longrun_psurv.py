"""Writes tests/golden/<cfg>_psurv_oracle.txt: the domain-averaged survival probability of a BASELINE workload
over its FULL run, computed by the CPU oracle only (oracle/, OpenMP over z), sampled every `--every` steps.

    python tests/golden/make_longrun_psurv.py --cfg cfg2 [--threads 6] [--every 100] [--steps N]

This is the stored expected value of tests/test_gpu_long.py::test_cfg2_full_run_against_stored_oracle_series
(BASELINE north_star: "domain-averaged survival probability must agree within 1e-6 over the full run").
No value in the output comes from the CUDA path.  Rows are appended and flushed as the run proceeds, so an
interrupted run leaves a valid (shorter) series.  A run that does not fit one session can stop itself after
--budget-s seconds, writing the ORACLE's state to --checkpoint, and be continued with --resume (same --out).

Cost: cfg2 (32768 x 128, WENO7, 5000 steps) is about 2.1e10 cell-steps: hours on a few host cores.
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import cosenu_ref as R                      # noqa: E402
from paper_2203_12866_b200 import inputs                # noqa: E402  (seeded input generators only)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", default="cfg2")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--every", type=int, default=100)
    ap.add_argument("--steps", type=int, default=0, help="0 = the workload's full length")
    ap.add_argument("--out", default="")
    ap.add_argument("--budget-s", type=float, default=0.0, help="stop after this many seconds (at a sample) and write --checkpoint")
    ap.add_argument("--checkpoint", default="", help=".npz to write when the budget is used up / to read with --resume")
    ap.add_argument("--resume", action="store_true", help="continue from --checkpoint, appending to --out")
    a = ap.parse_args()
    c = inputs.CONFIGS[a.cfg]
    nsteps = a.steps or c["steps"]
    out = a.out or os.path.join(ROOT, "tests", "golden", "%s_psurv_oracle.txt" % a.cfg)
    r = R.RefSim(c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"], threads=a.threads)
    # A resumed run re-uploads the oracle's own state (cosenu_ref_set_state), which re-takes the t = 0 references of the
    # diagnostics; the ratios to the true t = 0 are carried in the checkpoint: psurv(t) = [sum rho_ee(t) / sum rho_ee(t_c)] *
    # psurv(t_c), and M0(t) - M0(0) = [M0(t) - M0(t_c)] + [M0(t_c) - M0(0)].
    done, scale_nu, scale_nubar, dM0_base = 0, 1.0, 1.0, np.zeros(3)
    if a.resume:
        ck = np.load(a.checkpoint)
        r.set_state(ck["state"], float(ck["t"]))
        done, scale_nu, scale_nubar, dM0_base = int(ck["step"]), float(ck["psurv_nu"]), float(ck["psurv_nubar"]), ck["dM0"]
    else:
        r.set_state(inputs.config_state(a.cfg))
    t0 = time.time()
    with open(out, "a" if a.resume else "w") as f:
        if not a.resume:
            f.write("# Oracle-only time series of BASELINE %s (seed %d, %d x %d, scheme %d, dt %.17g): written by\n"
                    "# tests/golden/make_longrun_psurv.py --cfg %s --every %d ; <rho_ee>(t) of PAPER.md:229 (multi-angle\n"
                    "# reading R1 of DESIGN.md), max|rho_ex| and the largest |M0(t) - M0(0)| component (Eq. 19, PAPER.md:247).\n"
                    "# columns: step psurv_nu psurv_nubar ex_abs_max dM0_max\n"
                    % (a.cfg, c["seed"], c["nz"], c["nv"], c["scheme"], c["dt"], a.cfg, a.every))
        else:
            f.write("# resumed from the oracle's own checkpoint at step %d (same script, --resume)\n" % done)
        while done < nsteps:
            n = min(a.every, nsteps - done)
            r.step(n)
            done += n
            d = r.diagnostics()
            ps_nu, ps_nubar = d["psurv_nu"] * scale_nu, d["psurv_nubar"] * scale_nubar
            dM0 = np.array(d["dM0"]) + dM0_base
            f.write("%d %.17g %.17g %.17g %.17g\n" % (done, ps_nu, ps_nubar, d["ex_abs_max"], float(np.max(np.abs(dM0)))))
            f.flush()
            print("step %d  psurv_nu %.12f  ex_max %.3e  %.0f s" % (done, ps_nu, d["ex_abs_max"], time.time() - t0), flush=True)
            if a.budget_s and a.checkpoint and done < nsteps and time.time() - t0 > a.budget_s:
                np.savez(a.checkpoint, state=r.get_state(), t=d["t"], step=done, psurv_nu=ps_nu, psurv_nubar=ps_nubar, dM0=dM0)
                print("budget used up: checkpoint at step %d -> %s" % (done, a.checkpoint), flush=True)
                break
    r.close()


if __name__ == "__main__":
    main()
