"""Writes tests/golden/<cfg>_psurv_oracle.txt: the domain-averaged survival probability of a BASELINE workload
over its FULL run, computed by the CPU oracle only (oracle/, OpenMP over z), sampled every `--every` steps.

    python tests/golden/make_longrun_psurv.py --cfg cfg2 [--threads 6] [--every 100] [--steps N]

This is the stored expected value of tests/test_gpu_long.py::test_cfg2_full_run_against_stored_oracle_series
(BASELINE north_star: "domain-averaged survival probability must agree within 1e-6 over the full run").
No value in the output comes from the CUDA path.  Rows are appended and flushed as the run proceeds, so an
interrupted run leaves a valid (shorter) series; rerun with --resume to continue is NOT supported (the oracle
keeps its state in memory only) -- the header records how far the file goes.

Cost: cfg2 (32768 x 128, WENO7, 5000 steps) is about 2.1e10 cell-steps: hours on a few host cores.
"""
import argparse
import os
import sys
import time

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
    a = ap.parse_args()
    c = inputs.CONFIGS[a.cfg]
    nsteps = a.steps or c["steps"]
    out = a.out or os.path.join(ROOT, "tests", "golden", "%s_psurv_oracle.txt" % a.cfg)
    r = R.RefSim(c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"], threads=a.threads)
    r.set_state(inputs.config_state(a.cfg))
    t0 = time.time()
    with open(out, "w") as f:
        f.write("# Oracle-only time series of BASELINE %s (seed %d, %d x %d, scheme %d, dt %.17g): written by\n"
                "# tests/golden/make_longrun_psurv.py --cfg %s --every %d ; <rho_ee>(t) of PAPER.md:229 (multi-angle\n"
                "# reading R1 of DESIGN.md), max|rho_ex| and the largest |M0(t) - M0(0)| component (Eq. 19, PAPER.md:247).\n"
                "# columns: step psurv_nu psurv_nubar ex_abs_max dM0_max\n"
                % (a.cfg, c["seed"], c["nz"], c["nv"], c["scheme"], c["dt"], a.cfg, a.every))
        done = 0
        while done < nsteps:
            n = min(a.every, nsteps - done)
            r.step(n)
            done += n
            d = r.diagnostics()
            f.write("%d %.17g %.17g %.17g %.17g\n" % (d["step"], d["psurv_nu"], d["psurv_nubar"], d["ex_abs_max"],
                                                     max(abs(x) for x in d["dM0"])))
            f.flush()
            print("step %d  psurv_nu %.12f  ex_max %.3e  %.0f s" % (done, d["psurv_nu"], d["ex_abs_max"], time.time() - t0),
                  flush=True)
    r.close()


if __name__ == "__main__":
    main()
