"""Seeded random differential test: random shapes (ragged in z and v, odd N_v so that one 32-beam chunk holds both signs of v),
schemes, kernel shapes, RK carriers, quadrature rules, KO orders, physics parameters and slab cuts; two RK4 steps from a rough
O(1) state against the oracle, and the slab-decomposed run against the single domain bit for bit."""
import numpy as np
import pytest

from paper_2203_12866_b200 import inputs

pytestmark = pytest.mark.gpu


def _cases(n, seed):
    rng = np.random.default_rng(seed)
    out = []
    for k in range(n):
        scheme = int(rng.integers(0, 2))
        quad = int(rng.integers(0, 3))
        nv = int(rng.integers(2, 131))
        if quad == 2 and nv % 2 == 0:
            nv += 1
        nz = int(rng.integers(16, 420))
        nslabs = int(rng.integers(1, 5))
        while nz // nslabs < 16:
            nslabs -= 1
        cuts = sorted(rng.choice(np.arange(16, nz - 15), size=nslabs - 1, replace=False).tolist()) if nslabs > 1 else []
        edges = [0] + cuts + [nz]
        if any(b - a < 16 for a, b in zip(edges, edges[1:])):
            edges = [0, nz]
        out.append(dict(scheme=scheme, quad=quad, nv=nv, nz=nz, variant=int(rng.integers(0, 3)), rk_form=int(rng.integers(0, 4)),
                        ko=int(rng.choice([2, 3])) if scheme == 0 else 2, omega=float(rng.uniform(0, 1.5)),
                        theta=float(rng.uniform(0, 0.8)), mu=float(rng.uniform(0, 2.0)), dt=float(rng.uniform(0.01, 0.1)),
                        L=float(nz * rng.uniform(0.5, 2.0)), bounds=[(a, b - a) for a, b in zip(edges, edges[1:])], seed=1000 + k))
    return out


@pytest.mark.parametrize("case", _cases(48, 20221286), ids=lambda c: "nz%d-nv%d-s%d-v%d-f%d-q%d-k%d-slabs%d" % (
    c["nz"], c["nv"], c["scheme"], c["variant"], c["rk_form"], c["quad"], c["ko"], len(c["bounds"])))
def test_random_case_vs_oracle_and_slabs(case):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import cosenu_ref as R
    from paper_2203_12866_b200 import binding as B, slab as S
    c = case
    st = inputs.random_state(c["nz"], c["nv"], seed=c["seed"])
    args = (c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"])
    opts = dict(variant=c["variant"], rk_form=c["rk_form"], quadrature=c["quad"], ko_order=c["ko"])
    g = B.Cosenu(*args, **opts)
    g.set_state(st)
    g.step(2)
    got, gm = g.get_state(), g.get_moments()
    g.close()
    r = R.RefSim(*args, quadrature=c["quad"], ko_order=c["ko"])
    r.set_state(st)
    r.step(2)
    ref = r.get_state()
    rm = r.moments(ref)
    r.close()
    scale = max(1.0, float(np.max(np.abs(ref))))
    assert np.max(np.abs(got - ref)) <= 5e-14 * scale
    assert np.max(np.abs(gm - rm)) <= 2e-14 * max(1.0, float(np.max(np.abs(rm))))
    grp = S.SlabGroup(len(c["bounds"]), *args, bounds=c["bounds"], **opts)
    grp.set_state(st)
    grp.step(2)
    grp.sync()
    sl, slm = grp.get_state(), grp.get_moments()
    grp.close()
    assert np.array_equal(sl, got) and np.array_equal(slm, gm)
