"""z-slab decomposition on ONE device: several slabs of one periodic grid, driven by one process on one
stream (stage by stage, so that no kernel waits for a kernel queued behind it), against the single-domain solver and the
oracle.  The decomposed path uses exactly the multi-GPU code: edge rows stored into the neighbouring slab's ghost rows,
arrival counters, edge tiles first; only the peer mapping (same-process addresses instead of cudaIpcOpenMemHandle) differs.
"""
import numpy as np
import pytest

from paper_2203_12866_b200 import inputs

pytestmark = pytest.mark.gpu

FD, FV = 0, 1


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2203_12866_b200 import binding
    binding.load()
    return binding


@pytest.fixture(scope="module")
def S(B):
    from paper_2203_12866_b200 import slab
    return slab


def _single(B, args, st, nsteps, **opts):
    g = B.Cosenu(*args, **opts)
    g.set_state(st)
    g.step(nsteps)
    out = g.get_state(), g.get_moments(), g.diagnostics()
    g.close()
    return out


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("scheme", [FD, FV])
@pytest.mark.parametrize("nslabs,nz,nv", [(1, 200, 40), (2, 200, 40), (3, 200, 40), (2, 35, 5), (4, 5000, 33), (5, 16 * 5, 70)])
def test_slab_group_equals_single_domain(B, S, scheme, nslabs, nz, nv, variant):
    """Rough O(1) random state, 3 steps: the decomposed run reproduces the single-domain run bit for bit (same per-cell
    arithmetic, same summation order of the moments), for ragged slabs, slabs of one tile, and a slab linked to itself."""
    st = inputs.random_state(nz, nv, seed=500 + nz + nv)
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
    ref, refm, refd = _single(B, args, st, 3, variant=variant)
    grp = S.SlabGroup(nslabs, *args, variant=variant)
    grp.set_state(st)
    grp.step(3)
    grp.sync()
    got, gotm, gotd = grp.get_state(), grp.get_moments(), grp.diagnostics()
    grp.close()
    assert np.array_equal(got, ref)
    assert np.array_equal(gotm, refm)
    for k in ("psurv_nu", "psurv_nubar", "dP_avg"):
        assert abs(gotd[k] - refd[k]) <= 1e-13, k
    for k in ("dP_max", "trace_dev_max", "ex_abs_max"):
        assert abs(gotd[k] - refd[k]) <= 1e-13 * max(1.0, abs(refd[k])), k
    assert np.max(np.abs(np.array(gotd["M0"]) - np.array(refd["M0"]))) <= 1e-12
    assert gotd["step"] == 3 and abs(gotd["t"] - 0.15) < 1e-15


@pytest.mark.parametrize("scheme", [FD, FV])
@pytest.mark.parametrize("rk_form", [0, 1, 2, 3])
def test_slab_group_vs_oracle_20_steps(B, S, scheme, rk_form):
    """BASELINE config 0 recipe over 3 uneven slabs, 20 steps, all RK carriers, against the oracle (1e-12)."""
    from oracle import cosenu_ref as R
    c = inputs.CONFIGS["cfg0"]
    st = inputs.config_state("cfg0")
    args = (c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], scheme)
    grp = S.SlabGroup(3, *args, rk_form=rk_form, bounds=[(0, 100), (100, 600), (700, 324)])
    grp.set_state(st)
    grp.step(20)
    grp.sync()
    got = grp.get_state()
    gd = grp.diagnostics()
    grp.close()
    r = R.RefSim(*args)
    r.set_state(st)
    r.step(20)
    ref, rd = r.get_state(), r.diagnostics()
    r.close()
    assert np.max(np.abs(got - ref)) <= 1e-12
    assert abs(gd["psurv_nu"] - rd["psurv_nu"]) <= 1e-12
    assert max(abs(x) for x in gd["dM0"]) <= 1e-11


def test_slab_init_builds_the_global_state(B, S):
    """cosenu_init on slabs builds each slab's rows of the global seeded state (the splitmix64 stream is entered at
    z_begin), for all three perturbation kinds."""
    nz, nv = 700, 12
    for kind in (0, 1, 2):
        for scheme in (FD, FV):
            args = (nz, nv, float(nz), 0.4, 0.0, 0.0, 1.0, scheme)
            g = B.Cosenu(*args)
            g.init(12866, pert_amp=1e-2 if kind == 2 else 1e-6, pert_kind=kind)
            ref = g.get_state()
            g.close()
            grp = S.SlabGroup(3, *args)
            grp.init(12866, pert_amp=1e-2 if kind == 2 else 1e-6, pert_kind=kind)
            got = grp.get_state()
            d = grp.diagnostics()
            grp.close()
            assert np.array_equal(got, ref), (kind, scheme)
            assert abs(d["psurv_nu"] - 1.0) <= 1e-14


def test_slab_self_linked_rank(B, S):
    """CosenuSlab without torch.distributed = one slab linked to itself (the code path a 1-rank job takes)."""
    nz, nv = 300, 20
    st = inputs.fast_conversion_state(nz, nv, seed=11, pert_amp=1e-3)
    args = (nz, nv, float(nz), 0.4, 1e-2, 0.01, 1.0, FV)
    ref, refm, refd = _single(B, args, st, 10)
    s = S.CosenuSlab(*args)
    assert (s.world, s.rank, s.z_begin, s.nz) == (1, 0, 0, nz)
    s.set_state(st)
    s.step(10)
    s.sync()
    assert np.array_equal(s.get_state(), ref)
    d = s.diagnostics()
    assert abs(d["psurv_nu"] - refd["psurv_nu"]) <= 1e-13
    s.close()


def test_slab_call_order_errors(B, S):
    h = B.Cosenu(64, 8, 64.0, 0.1, 0, 0, 1.0, FD, use_torch_workspace=False, slab=(128, 0))
    h.set_state(inputs.random_state(64, 8, seed=1))
    with pytest.raises(B.CosenuError) as e:
        h.step(1)                                   # not linked, ghosts not exchanged
    assert e.value.code == B.ESTATE
    with pytest.raises(B.CosenuError) as e:
        h.diagnostics()                             # a slab holds part of the grid
    assert e.value.code == B.ESTATE
    h.close()
    with pytest.raises(B.CosenuError):
        B.Cosenu(8, 8, 64.0, 0.1, 0, 0, 1.0, FD, slab=(128, 0))        # thinner than 16 rows
    with pytest.raises(B.CosenuError):
        B.Cosenu(64, 8, 64.0, 0.1, 0, 0, 1.0, FD, slab=(32, 0))        # larger than the grid
    with pytest.raises(B.CosenuError):
        B.Cosenu(64, 8, 64.0, 0.1, 0, 0, 1.0, FD, slab=(128, 100))     # sticks out of the grid


# ---------------------------------------------------------------------------------------------------------
# The cross-PROCESS leg (cudaIpcGetMemHandle / cudaIpcOpenMemHandle, peer stores and counters in another process's
# memory): two ranks share the one GPU, driven in lockstep (sync + barrier after every stage), so no kernel ever waits for
# a kernel of the other process -- every counter has arrived before the launch that checks it.
def _ipc_worker(rank, world, port, nz, nv, scheme, nsteps, q):
    import os
    import sys
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import torch
    import torch.distributed as dist
    from paper_2203_12866_b200 import inputs as I, slab as S
    torch.cuda.set_device(0)
    import datetime
    dist.init_process_group("gloo", rank=rank, world_size=world, timeout=datetime.timedelta(seconds=90))
    try:
        st = I.random_state(nz, nv, seed=900 + nz + nv)
        s = S.CosenuSlab(nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
        s.set_state(np.ascontiguousarray(st[:, s.z_begin:s.z_begin + s.nz, :]))
        s.step_lockstep(nsteps)
        s.sync()
        d = s.diagnostics()
        q.put((rank, s.z_begin, s.nz, s.get_state(), d))
        s.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("scheme,world", [(FD, 2), (FV, 2), (FV, 3)])
def test_slabs_in_separate_processes_over_cuda_ipc(B, scheme, world):
    import torch.multiprocessing as mp
    nz, nv, nsteps = 150, 40, 3
    st = inputs.random_state(nz, nv, seed=900 + nz + nv)
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
    ref, _, refd = _single(B, args, st, nsteps)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    from conftest import free_port
    port = free_port()
    ps = [ctx.Process(target=_ipc_worker, args=(r, world, port, nz, nv, scheme, nsteps, q)) for r in range(world)]
    for p in ps:
        p.start()
    try:
        outs = sorted((q.get(timeout=200) for _ in ps), key=lambda o: o[0])
        for p in ps:
            p.join(120)
            assert p.exitcode == 0
    finally:
        for p in ps:
            if p.is_alive():
                p.terminate()
    got = np.concatenate([o[3] for o in outs], axis=1)
    assert [o[1] for o in outs][0] == 0 and sum(o[2] for o in outs) == nz
    assert np.array_equal(got, ref)
    for o in outs:
        assert abs(o[4]["psurv_nu"] - refd["psurv_nu"]) <= 1e-13 and o[4]["step"] == nsteps


# ------------------------------------------------------------------ the halo-exchange protocol under real concurrency
def _sm_count():
    import torch
    return torch.cuda.get_device_properties(0).multi_processor_count


@pytest.mark.parametrize("scheme", [FD, FV])
@pytest.mark.parametrize("nslabs,skew", [(2, None), (2, (0.0, 0.3)), (2, (0.3, 0.0)), (3, None), (3, (0.2, 0.0, 0.1))])
def test_free_running_slabs_spin_on_each_other(B, S, scheme, nslabs, skew):
    """Every slab on its own stream, driven by its own host thread with the free-running cosenu_step(n); the persistent grid
    of every stage launch is capped (COSENU_OPT_MAX_CTAS) so that the kernels of all slabs are co-resident (one CTA per SM
    each) and nothing but the arrival counters orders them: the RAW wait and the WAR argument of DESIGN.md section 8 with
    kernels that really wait for each other -- also when one rank starts late.  Bit-identical to the single domain."""
    cap = _sm_count() // nslabs
    tiles_per_cta = 2
    nz = nslabs * cap * 16 * tiles_per_cta + (16 * 3 if nslabs == 3 else 0)     # every slab fills its capped grid; 3 slabs: ragged
    nv = 64
    st = inputs.random_state(nz, nv, seed=900 + nslabs)
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
    ref, refm, _ = _single(B, args, st, 12)
    grp = S.ConcurrentSlabs(nslabs, *args, max_ctas=cap)
    grp.set_state(st)
    grp.step(12, delays=skew)
    grp.sync()                       # raises if any halo wait timed out
    got, gotm = grp.get_state(), grp.get_moments()
    grp.close()
    assert np.array_equal(got, ref)
    assert np.array_equal(gotm, refm)


@pytest.mark.parametrize("scheme", [FD, FV])
def test_free_running_slabs_on_blocking_streams(B, S, scheme):
    """As above, but every handle owns a plain cudaStreamCreate stream (blocking: it synchronises with the legacy default
    stream), and slab 0's thread looks at every step (step(1) + sync) while slab 1 free-runs.  Nothing the library does
    between two launches may touch the legacy stream: it would wait for the other slab's queued stages, which spin on the
    stage this thread has not launched yet, until their halo wait times out (a spurious ESTATE)."""
    cap = _sm_count() // 2
    nz, nv = 2 * cap * 16 * 2, 64
    st = inputs.random_state(nz, nv, seed=911)
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
    ref, refm, _ = _single(B, args, st, 12)
    grp = S.ConcurrentSlabs(2, *args, max_ctas=cap, blocking_streams=True)
    grp.set_state(st)
    grp.step(12, sync_every_step=(True, False))
    grp.sync()
    got, gotm = grp.get_state(), grp.get_moments()
    grp.close()
    assert np.array_equal(got, ref)
    assert np.array_equal(gotm, refm)


def test_missing_neighbour_is_an_error_not_a_hang(B, S):
    """One slab of two steps alone: its waits give up, the flag is raised, and every call that hands results out reports it."""
    nz, nv = 2 * 16 * 8, 32
    st = inputs.random_state(nz, nv, seed=77)
    grp = S.ConcurrentSlabs(2, nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, FV, max_ctas=8)
    grp.set_state(st)
    grp.sims[0].step(1)              # slab 1 never steps: stage 2 of slab 0 waits for rows that never come
    with pytest.raises(B.CosenuError):
        grp.sims[0].sync()
    assert S._wait_failed(grp.sims[0])
    with pytest.raises(B.CosenuError):
        grp.sims[0].get_state()
    for s in grp.sims:
        s.close()
    grp.sims = []


def test_halo_timeout_is_an_option(B, S):
    """COSENU_OPT_HALO_TIMEOUT_S: with 0.5 s a slab whose neighbour never steps is flagged well before the default 4 s."""
    import time
    nz, nv = 2 * 16 * 8, 32
    grp = S.ConcurrentSlabs(2, nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, FV, max_ctas=8)
    for s in grp.sims:
        s.set_option(B.OPT_HALO_TIMEOUT_S, 0.5)
    for bad in (0.0, -1.0, 1e6, float("nan")):
        with pytest.raises(B.CosenuError):
            grp.sims[0].set_option(B.OPT_HALO_TIMEOUT_S, bad)
    grp.set_state(inputs.random_state(nz, nv, seed=78))
    t0 = time.perf_counter()
    grp.sims[0].step(1)
    with pytest.raises(B.CosenuError):
        grp.sims[0].sync()
    assert time.perf_counter() - t0 < 3.0
    assert S._wait_failed(grp.sims[0])
    for s in grp.sims:
        s.close()
    grp.sims = []


def test_two_gpus_free_running(B, S):
    """Two slabs on two GPUs of this process (peer access), free-running: needs a box with at least two devices."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    nz, nv = 2 * 148 * 16, 64
    st = inputs.random_state(nz, nv, seed=31)
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, FV)
    ref, refm, _ = _single(B, args, st, 10)
    bounds = [S.slab_bounds(nz, 2, r) for r in range(2)]
    sims = []
    for d, (zb, nzl) in enumerate(bounds):
        with torch.cuda.device(d):
            sims.append(B.Cosenu(nzl, nv, *args[2:], use_torch_workspace=False, stream=torch.cuda.Stream(device=d), slab=(nz, zb)))
    peers = [S._export(s) for s in sims]
    for r, s in enumerate(sims):
        S._link(s, peers[(r - 1) % 2], peers[(r + 1) % 2])
    grp = S.ConcurrentSlabs.__new__(S.ConcurrentSlabs)
    grp.nz_global, grp.nv, grp.bounds, grp.sims, grp._L = nz, nv, bounds, sims, sims[0]._L
    grp.set_state(st)
    grp.step(10)
    grp.sync()
    got = grp.get_state()
    grp.close()
    assert np.array_equal(got, ref)
