"""CPU-only checks of the product's host side: the C-ABI library loads without a GPU and exports every
symbol include/cosenu.h declares; it fails loudly (no CPU fallback); the stencil arithmetic the kernels use
(csrc/weno7_math.h, host build) agrees with the oracle's literal App. A formulas."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2203_12866_b200 import build as pbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libs():
    import build_probe
    pbuild.build()
    return C.CDLL(pbuild.LIB), C.CDLL(build_probe.build())


def test_library_exports_every_declared_symbol(libs):
    lib, _ = libs
    hdr = open(os.path.join(ROOT, "include", "cosenu.h")).read()
    declared = sorted(set(re.findall(r"\b(cosenu_[a-z_0-9]+)\s*\(", hdr)))
    from paper_2203_12866_b200 import binding
    assert sorted(binding.SYMBOLS) == declared
    for s in declared:
        assert getattr(lib, s) is not None


def test_no_cpu_fallback_without_gpu(libs):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2203_12866_b200 import binding
    with pytest.raises(binding.CosenuError) as e:
        binding.Cosenu(64, 4, 1.0, 0.1, 0.0, 0.0, 0.0, 0, use_torch_workspace=False)
    assert "CUDA" in str(e.value)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2203_12866_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dp, f)).read()
                assert "cosenu_ref" not in txt and "import oracle" not in txt and "from oracle" not in txt, f


def test_kernel_weno_formula_matches_oracle_algorithm1(libs):
    from oracle import cosenu_ref as R
    _, probe = libs
    dp = C.POINTER(C.c_double)
    probe.cosenu_probe_weno7_face.restype = C.c_double
    probe.cosenu_probe_weno7_face.argtypes = [dp, C.c_double, C.c_double]
    rng = np.random.default_rng(20221286)
    for trial in range(4000):
        kind = trial % 3
        if kind == 0:
            w = rng.standard_normal(7)                    # rough O(1)
        elif kind == 1:
            w = np.sin(0.3 * np.arange(7) + rng.uniform(0, 6))   # smooth
        else:
            w = 1e-6 * rng.standard_normal(7)             # tiny (SI << eps: linear weights)
        v = rng.uniform(-1, 1)
        for eps in (1e-6, 1e30):
            a = probe.cosenu_probe_weno7_face(w.ctypes.data_as(dp), v, eps)
            b = R.weno7_face(v * w, eps)
            assert abs(a - b) <= 5e-14 * np.max(np.abs(v * w)) + 1e-300


def test_kernel_fd_formula_matches_definition_and_is_exact_on_constants(libs):
    _, probe = libs
    dp = C.POINTER(C.c_double)
    probe.cosenu_probe_fd4_ko3.restype = C.c_double
    probe.cosenu_probe_fd4_ko3.argtypes = [dp, C.c_double, C.c_double, C.c_double]
    rng = np.random.default_rng(5)
    for _ in range(1000):
        u = rng.standard_normal(5); v = rng.uniform(-1, 1); dz = rng.uniform(0.1, 2); ek = rng.uniform(0, 1)
        a = probe.cosenu_probe_fd4_ko3(u.ctypes.data_as(dp), v, dz, ek)
        b = -v * (u[0] - 8 * u[1] + 8 * u[3] - u[4]) / (12 * dz) - (ek / (16 * dz)) * (u[0] - 4 * u[1] + 6 * u[2] - 4 * u[3] + u[4])
        assert abs(a - b) <= 1e-14 / dz
    u = np.full(5, 0.7331)
    assert probe.cosenu_probe_fd4_ko3(u.ctypes.data_as(dp), 0.9, 1.0, 0.1) == 0.0
    # Kreiss-Oliger r = 3 (Eq. 5): eps h^5 (D+ D-)^3 / 64 with the dissipative sign = + (eps/64dz) delta^6 u
    probe.cosenu_probe_fd4_ko5.restype = C.c_double
    probe.cosenu_probe_fd4_ko5.argtypes = [dp, C.c_double, C.c_double, C.c_double]
    for _ in range(1000):
        u = rng.standard_normal(7); v = rng.uniform(-1, 1); dz = rng.uniform(0.1, 2); ek = rng.uniform(0, 1)
        a = probe.cosenu_probe_fd4_ko5(u.ctypes.data_as(dp), v, dz, ek)
        d6 = u[0] - 6 * u[1] + 15 * u[2] - 20 * u[3] + 15 * u[4] - 6 * u[5] + u[6]
        b = -v * (u[1] - 8 * u[2] + 8 * u[4] - u[5]) / (12 * dz) + (ek / (64 * dz)) * d6
        assert abs(a - b) <= 2e-14 / dz
    u = np.full(7, 0.7331)
    assert probe.cosenu_probe_fd4_ko5(u.ctypes.data_as(dp), 0.9, 1.0, 0.1) == 0.0
    u = (-1.0) ** np.arange(7)          # Nyquist mode: Q u = -(eps/dz) u at the centre cell (u_3 = -1)
    assert abs(probe.cosenu_probe_fd4_ko5(u.ctypes.data_as(dp), 0.3, 1.0, 0.1) - 0.1) <= 1e-16


def test_kernel_weno_form_against_exact_rational_algorithm1(libs):
    """Algorithm 1 in exact rational arithmetic is the judge between the two fp64 evaluation
    orders: the oracle's literal Eq. (A.3) polynomials and the kernels' difference form.  Both must agree with it;
    for nearly constant O(1) data the literal form loses digits, the difference form must not."""
    from fractions import Fraction as F
    from oracle import cosenu_ref as R
    _, probe = libs
    dp = C.POINTER(C.c_double)
    probe.cosenu_probe_weno7_face.restype = C.c_double
    probe.cosenu_probe_weno7_face.argtypes = [dp, C.c_double, C.c_double]
    probe.cosenu_probe_weno7_face2.restype = None
    probe.cosenu_probe_weno7_face2.argtypes = [dp, C.c_double, C.c_double, dp]

    def exact(f, eps):
        m3, m2, m1, c, p1, p2, p3 = [F(x) for x in f]
        fh = [(3 * c + 13 * p1 - 5 * p2 + p3) / 12, (-m1 + 7 * c + 7 * p1 - p2) / 12,
              (m2 - 5 * m1 + 13 * c + 3 * p1) / 12, (-3 * m3 + 13 * m2 - 23 * m1 + 25 * c) / 12]
        si = [c * (2107 * c - 9402 * p1 + 7042 * p2 - 1854 * p3) + p1 * (11003 * p1 - 17246 * p2 + 4642 * p3)
              + p2 * (7043 * p2 - 3882 * p3) + 547 * p3 * p3,
              m1 * (547 * m1 - 2522 * c + 1922 * p1 - 494 * p2) + c * (3443 * c - 5966 * p1 + 1602 * p2)
              + p1 * (2843 * p1 - 1642 * p2) + 267 * p2 * p2,
              m2 * (267 * m2 - 1642 * m1 + 1602 * c - 494 * p1) + m1 * (2843 * m1 - 5966 * c + 1922 * p1)
              + c * (3443 * c - 2522 * p1) + 547 * p1 * p1,
              m3 * (547 * m3 - 3882 * m2 + 4642 * m1 - 1854 * c) + m2 * (7043 * m2 - 17246 * m1 + 7042 * c)
              + m1 * (11003 * m1 - 9402 * c) + 2107 * c * c]
        d = [F(4, 35), F(18, 35), F(12, 35), F(1, 35)]
        w = [d[r] / (si[r] + F(eps)) ** 2 for r in range(4)]
        return sum(w[r] * fh[r] for r in range(4)) / sum(w)

    rng = np.random.default_rng(7)
    worst_kernel, worst_oracle = 0.0, 0.0
    for trial in range(300):
        kind = trial % 3
        if kind == 0:
            u = rng.standard_normal(8)
        elif kind == 1:
            u = 1.0 + 1e-3 * rng.standard_normal(8)          # nearly constant O(1): the cancellation case
        else:
            u = np.sin(0.25 * np.arange(8) + rng.uniform(0, 6))
        v, eps = float(rng.uniform(0.05, 1.0)), 1e-6
        f = [v * x for x in u]                                # Algorithm 1 acts on f = v u (reading A8)
        ex = exact(f[:7], eps)
        a = probe.cosenu_probe_weno7_face(u[:7].copy().ctypes.data_as(dp), v, eps)
        o = R.weno7_face(np.array(f[:7]), eps)
        scale = max(abs(x) for x in f)
        ek, eo = abs(F(a) - ex) / F(scale), abs(F(o) - ex) / F(scale)
        worst_kernel, worst_oracle = max(worst_kernel, float(ek)), max(worst_oracle, float(eo))
        # the paired routine gives the same two interfaces as two single calls
        out = np.empty(2)
        probe.cosenu_probe_weno7_face2(u.ctypes.data_as(dp), v, eps, out.ctypes.data_as(dp))
        b = probe.cosenu_probe_weno7_face(u[1:8].copy().ctypes.data_as(dp), v, eps)
        assert abs(out[0] - a) <= 4e-16 * scale and abs(out[1] - b) <= 4e-16 * scale
    assert worst_kernel <= 2e-15, worst_kernel     # the kernels' form is accurate to a few ulp everywhere
    assert worst_oracle <= 5e-11, worst_oracle     # the literal form is right too, up to its cancellation noise


def test_analysis_dP_map_matches_the_diagnostics_definition():
    """analysis.dP_map (Fig. 10's delta P(z,v)) against Eq. (22) as the oracle's diagnostics take it."""
    from oracle import cosenu_ref as R
    from paper_2203_12866_b200 import analysis, inputs
    c = inputs.CONFIGS["cfg0"]
    st0 = inputs.config_state("cfg0")
    r = R.RefSim(c["nz"], c["nv"], c["L"], c["dt"], 0.0, 0.0, 1.0, 0)
    r.set_state(st0)
    r.step(150)
    d = r.diagnostics()
    m = max(np.abs(analysis.dP_map(r.get_state(), st0, s)).max() for s in (0, 1))
    assert abs(m - d["dP_max"]) <= 1e-13
    assert analysis.dP_map(st0, st0).max() <= 1e-12      # 1e-6 seed: |P| is uniform in z to O(1e-12) at t = 0
    r.close()


def test_analysis_estimators_on_known_sequences():
    """E2 (Eq. 15), kappa (Eq. 24) and the three-error order estimator (Eq. C.3) as printed, on
    sequences whose answers are known; plus the two textbook estimators that keep their own names."""
    from paper_2203_12866_b200 import analysis
    assert abs(analysis.e2_norm([1.0, 2.0, 3.0], [1.0, 2.0, 5.0]) - np.sqrt(4.0 / 3.0)) < 1e-15
    # Eq. (24): dP_max halves four times when N_z doubles -> kappa = 4; equal errors (time-integration floor) -> kappa = 0
    assert analysis.kappa(3.2e-3, 2.0e-4) == pytest.approx(4.0, abs=1e-12)
    assert analysis.kappa(2.5e-13, 2.5e-13) == 0.0
    assert analysis.kappa(1.0, 8.0) == pytest.approx(-3.0, abs=1e-12)
    for p in (3.0, 4.0, 7.0):
        # Eq. (C.2): E_i = C_z (dz_0 / r^i)^alpha + C_t dt^beta with one dt for all i: the constant cancels in Eq. (C.3)
        for r in (2.0, 3.0):
            E = [0.7 * (0.4 / r ** i) ** p + 0.123 for i in range(3)]
            assert abs(analysis.order_of_convergence(*E, ratio=r) - p) < 1e-9
        # whereas the two-error ratio is fooled by that constant, and exact without it
        assert abs(analysis.two_grid_order(5.0, 5.0 / 2 ** p) - p) < 1e-12
        assert analysis.two_grid_order(5.0 + 0.123, 5.0 / 2 ** p + 0.123) < p - 0.05
        q = [1.0 + 0.3 * h ** p for h in (0.4, 0.2, 0.1)]                                   # q(h) = q* + C h^p
        assert abs(analysis.richardson_ratio(*q) - 2 ** p) < 1e-6 * 2 ** p
    assert analysis.richardson_ratio(1.0, 2.0, 2.0) == float("inf")


def test_oracle_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """SURVEY.md section 5 (race detection / sanitizers): the oracle built with -fsanitize=address,undefined runs the FD closed
    form (P3), the WENO linear limit (P6) and the brute-force commutator / moments (P9) pins without a report.  The sanitized
    library is loaded in a child process (ASan must be the first DSO), which runs those pins of tests/test_oracle_pins.py."""
    import shutil
    import subprocess
    import sys
    if shutil.which("g++") is None:
        pytest.skip("no g++")
    out = tmp_path / "libcosenu_ref_asan.so"
    src = os.path.join(ROOT, "oracle", "cosenu_ref.cpp")
    r = subprocess.run(["g++", "-std=c++17", "-O1", "-g", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                        "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
                        "-o", str(out), src], capture_output=True, text=True)
    if r.returncode != 0 and "sanitize" in (r.stderr or ""):
        pytest.skip("this g++ has no sanitizer runtime: " + r.stderr[-200:])
    assert r.returncode == 0, r.stderr
    asan = subprocess.run(["g++", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan):
        pytest.skip("libasan.so not found")
    env = dict(os.environ, LD_PRELOAD=asan, COSENU_REF_LIB=str(out),
               ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=0", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                        os.path.join(ROOT, "tests", "test_oracle_pins.py"),
                        "-k", "P3_fd_ko_discrete_closed_form or P6_weno_linear_limit or P9_commutator or diagnostics_hand_values"],
                       capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    tail = (r.stdout or "")[-1500:] + (r.stderr or "")[-1500:]
    assert r.returncode == 0, tail
    assert "ERROR: AddressSanitizer" not in tail and "runtime error" not in tail, tail
    assert "passed" in r.stdout
