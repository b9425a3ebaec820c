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
    pbuild.build()
    return C.CDLL(pbuild.LIB), C.CDLL(pbuild.PROBE)


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
