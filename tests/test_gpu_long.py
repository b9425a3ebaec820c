"""Long-run agreement of the domain-averaged survival probability (BASELINE north_star: within 1e-6 over the
full run) on config 0's full 500 steps, both schemes, sampled every 50 steps; the element-wise state difference
at the end is reported against the amplification of rounding by the unstable modes."""
import numpy as np
import pytest

from paper_2203_12866_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("scheme", [0, 1])
def test_cfg0_full_run_survival_probability(scheme):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import cosenu_ref as R
    from paper_2203_12866_b200 import binding as B
    c = inputs.CONFIGS["cfg0"]
    st = inputs.config_state("cfg0")
    args = (c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], scheme)
    g = B.Cosenu(*args)
    r = R.RefSim(*args)
    g.set_state(st)
    r.set_state(st)
    worst = 0.0
    for _ in range(c["steps"] // 50):
        g.step(50)
        r.step(50)
        dg, dr = g.diagnostics(), r.diagnostics()
        worst = max(worst, abs(dg["psurv_nu"] - dr["psurv_nu"]), abs(dg["psurv_nubar"] - dr["psurv_nubar"]))
        assert dg["step"] == dr["step"]
    assert worst <= 1e-6, worst
    # linear phase: rounding differences grow with the instability (x ~2000 over 500 steps)
    err = float(np.max(np.abs(g.get_state() - r.get_state())))
    assert err <= 1e-9, err
    assert max(abs(x) for x in dg["dM0"]) <= 1e-10      # M0 conserved to rounding
    g.close(); r.close()


def _read_series(path):
    rows = []
    with open(path) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                p = line.split()
                rows.append((int(p[0]), float(p[1]), float(p[2]), float(p[3]), float(p[4])))
    return rows


# Step up to which the GPU run and the oracle agree to 1e-6 in the domain-averaged survival probability on BASELINE
# config 2 (measured on B200, long runs).  Beyond it both runs are deep in the nonlinear regime,
# where rounding-level differences between two correct fp64 evaluations are amplified at the instability's own rate.
CFG2_AGREE_UNTIL = None    # None: the whole stored series


def test_cfg2_long_run_against_stored_oracle_series():
    """BASELINE config 2 (WENO7, 32768 x 128) against the oracle's stored time series
    (tests/golden/cfg2_psurv_oracle.txt, written by tests/golden/make_longrun_psurv.py from oracle/ only)."""
    import os
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg2_psurv_oracle.txt")
    if not os.path.exists(path):
        pytest.skip("stored oracle series not present")
    series = _read_series(path)
    assert len(series) >= 10
    from paper_2203_12866_b200 import binding as B
    c = inputs.CONFIGS["cfg2"]
    g = B.Cosenu(c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"])
    g.set_state(inputs.config_state("cfg2"))
    done, worst, first_bad, report = 0, 0.0, None, []
    for step, ps_nu, ps_nubar, ex_max, dm0 in series:
        g.step(step - done)
        done = step
        d = g.diagnostics()
        err = max(abs(d["psurv_nu"] - ps_nu), abs(d["psurv_nubar"] - ps_nubar))
        report.append((step, err, d["psurv_nu"]))
        if CFG2_AGREE_UNTIL is None or step <= CFG2_AGREE_UNTIL:
            worst = max(worst, err)
        if err > 1e-6 and first_bad is None:
            first_bad = step
        assert max(abs(x) for x in d["dM0"]) <= 1e-9 * c["nz"]        # M0 conserved, any length
    g.close()
    print("cfg2 long run: last step %d, worst |dPsurv| in the asserted range %.3e, first step above 1e-6: %s"
          % (done, worst, first_bad))
    print("  step, |dPsurv|, Psurv_gpu: " + "; ".join("%d %.2e %.6f" % r for r in report[::max(1, len(report) // 12)]))
    assert worst <= 1e-6, (worst, first_bad)


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_bandwidth_scale_configs_over_their_full_length(name):
    """BASELINE configs 3 (200 steps) and 4 (100 steps) at full size: what must hold at any size and length --
    the trace of every cell stays put (the commutator is traceless, the initial state is z-homogeneous), the lepton-number
    vector M0 is conserved (its projection on B-hat when the vacuum term is on, PAPER.md:247-249 / DESIGN R2), the
    survival probability stays in [0, 1], no NaN; and the state is reproduced bit for bit by a second run."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2203_12866_b200 import binding as B
    c = inputs.CONFIGS[name]
    free, _ = torch.cuda.mem_get_info()
    if free < 5 * 64 * c["nz"] * c["nv"]:
        pytest.skip("not enough device memory")
    out = []
    for _ in range(2):
        g = B.Cosenu(c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"])
        g.init(c["seed"])
        g.step(c["steps"])
        d = g.diagnostics()
        m = g.get_moments()
        g.close()
        out.append((d, m))
    d, m = out[0]
    assert d["step"] == c["steps"] and np.isfinite(m).all()
    assert d["trace_dev_max"] <= 1e-12
    assert 0.0 < d["psurv_nu"] <= 1.0 + 1e-12 and 0.0 < d["psurv_nubar"] <= 1.0 + 1e-12
    s2, c2 = np.sin(2 * c["theta"]), np.cos(2 * c["theta"])
    along_B = s2 * d["dM0"][0] - c2 * d["dM0"][2]
    assert abs(along_B) <= 1e-9 * c["nz"]
    if c["omega"] == 0.0:
        assert max(abs(x) for x in d["dM0"]) <= 1e-9 * c["nz"]
    assert np.array_equal(m, out[1][1]) and d == out[1][0]          # deterministic summation order: bitwise repeatable
