"""cosenu_beam_sums_static: the one entry point of the library that allocates no device memory.

Why it exists.  Every other call works on a handle, and a handle needs a workspace that somebody cudaMallocs.  Two
kinds of caller of this library cannot do that at the place where they want a diagnostic:
  * code running in a process whose pooling allocator (torch's caching allocator, RMM, ...) already owns the GPU's
    memory -- next to a 34 GB solver workspace a raw cudaMalloc fails or goes behind the pool's back;
  * code running beside free-running z-slab handles: cudaFree (and possibly cudaMalloc) waits for the whole device, the
    host thread stuck in it cannot enqueue its slab's next stage, and the neighbour's halo wait runs into its 4 s
    time-out, which invalidates the run.
The entry point therefore keeps its per-block partial sums in an array that is part of the library image (148 x 4 x 512
doubles, 2.3 MiB per GPU, shared by all calls, never cleared, never freed).

What is checked: the new call against the existing handle-based path (set_state -> diag_ref_kernel with workspace scratch ->
host sum, reached through cosenu_slab_ref_sums), at the relative tolerance the suite uses elsewhere (1e-14), on two
calls issued back to back on one stream with different sizes, so that whatever the first call leaves in the shared array
would show up in the second if it were ever read; then the first call again (must reproduce its own bits), the
largest v-grid the array holds, and the refusals.  Nothing here depends on which tests ran before: the address look-up
the first call does on a device works the same in a fresh process and in one that has used the library for minutes.
This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests).
"""
import ctypes as C

import numpy as np
import pytest

RTOL = 1e-14   # the suite's relative tolerance (test_gpu_parity.py: the init recipe check)


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2203_12866_b200 import binding
    binding.load()
    return binding


def _state(nz, nv, seed):
    """All eight components independent (a swapped component or beam index changes the sums), ee and xx positive so
    that no per-beam sum cancels; the sums do not need a physical state."""
    rng = np.random.default_rng(seed)
    st = rng.uniform(-0.5, 0.5, size=(8, nz, nv))
    st[[0, 1, 4, 5]] = rng.uniform(0.1, 1.0, size=(4, nz, nv))
    return st


def _existing_path(B, st):
    """The handle-based route: workspace scratch, partial sums added on the host."""
    from paper_2203_12866_b200 import slab
    _, nz, nv = st.shape
    sim = B.Cosenu(nz, nv, float(nz), 0.4, 0.0, 0.0, 1.0, B.FD4_KO3)
    sim.set_state(st)
    out = slab._ref_sums(sim).reshape(4, nv).copy()
    sim.close()
    return out


def _definition(st):
    """out[4][nv] written out from include/cosenu.h's statement of the result, in numpy."""
    out = []
    for s in (0, 4):
        ee, xx, re, im = st[s], st[s + 1], st[s + 2], st[s + 3]
        out.append(np.sqrt((ee - xx) ** 2 + 4.0 * (re * re + im * im)).sum(axis=0))
        out.append((ee + xx).sum(axis=0))
    return np.stack(out)


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_handle_path(B):
    import torch
    # call 1: 4099 rows do not divide by the 148 z-ranges, 300 beams = one full group of 256 lanes + a ragged one;
    # call 2: fewer rows than z-ranges (48 blocks have nothing to sum) and fewer beams, so most of the array still
    #         holds call 1's partials when call 2 runs
    cases = [(4099, 300, 11), (100, 33, 12)]
    states = [_state(*c) for c in cases]
    dev_in = [torch.from_numpy(s).cuda() for s in states]
    dev_out = [torch.full((4, s.shape[2]), float("nan"), dtype=torch.float64, device="cuda") for s in states]
    torch.cuda.synchronize()
    B.beam_sums_static(dev_in[0], dev_out[0])     # back to back on the current stream, no wait in between
    B.beam_sums_static(dev_in[1], dev_out[1])
    torch.cuda.synchronize()
    got = [o.cpu().numpy() for o in dev_out]
    for st, g in zip(states, got):
        ref = _existing_path(B, st)
        assert np.all(np.isfinite(g))
        np.testing.assert_allclose(g, ref, rtol=RTOL, atol=0.0)
        np.testing.assert_allclose(g, _definition(st), rtol=1e-12, atol=0.0)
    # call 1 once more, after call 2 has overwritten part of the array: bit for bit what it gave the first time
    again = torch.full_like(dev_out[0], float("nan"))
    B.beam_sums_static(dev_in[0], again)
    torch.cuda.synchronize()
    assert np.array_equal(again.cpu().numpy(), got[0])


@pytest.mark.gpu
def test_largest_v_grid_and_a_side_stream(B):
    import torch
    nv = B.STATIC_MAX_NV
    st = _state(64, nv, 13)
    d_in = torch.from_numpy(st).cuda()
    d_out = torch.full((4, nv), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    B.beam_sums_static(d_in, d_out, stream=side)
    side.synchronize()
    np.testing.assert_allclose(d_out.cpu().numpy(), _existing_path(B, st), rtol=RTOL, atol=0.0)


@pytest.mark.gpu
def test_refusals_launch_nothing(B):
    import torch
    L = B.load()
    nv = B.STATIC_MAX_NV + 1
    d_in = torch.zeros((8, 16, nv), dtype=torch.float64, device="cuda")
    d_out = torch.full((4, nv), float("nan"), dtype=torch.float64, device="cuda")
    with pytest.raises(B.CosenuError) as e:
        B.beam_sums_static(d_in, d_out)
    assert e.value.code == B.EINVAL and str(B.STATIC_MAX_NV) in str(e.value) and "COSENU_STATIC_MAX_NV" in str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.isnan(d_out).all())          # nothing was launched
    # a host buffer where a device buffer belongs: refused up front instead of faulting in the kernel
    host = np.zeros((8, 16, 4))
    d_small = torch.zeros((4, 4), dtype=torch.float64, device="cuda")
    rc = L.cosenu_beam_sums_static(host.ctypes.data, 16, 4, d_small.data_ptr(), None)
    assert rc == B.EINVAL and b"host pointer" in L.cosenu_beam_sums_static_error()
    rc = L.cosenu_beam_sums_static(d_in.data_ptr(), 0, 4, d_small.data_ptr(), None)
    assert rc == B.EINVAL and b"nz" in L.cosenu_beam_sums_static_error()
    torch.cuda.synchronize()                        # and the device is still healthy
    B.beam_sums_static(torch.from_numpy(_state(16, 4, 14)).cuda(), d_small)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(d_small).all())


def test_size_limit_is_checked_before_any_cuda_call():
    """Runs without a GPU too: the limit is refused with its name in the text; with valid sizes and no device the call
    fails loudly (COSENU_ECUDA), it never computes anything on the CPU."""
    import torch
    from paper_2203_12866_b200 import binding as Bn
    L = Bn.load()
    rc = L.cosenu_beam_sums_static(None, 16, Bn.STATIC_MAX_NV + 1, None, None)
    assert rc == Bn.EINVAL and b"COSENU_STATIC_MAX_NV" in L.cosenu_beam_sums_static_error()
    if not torch.cuda.is_available():
        buf = (C.c_double * 64)()
        rc = L.cosenu_beam_sums_static(C.addressof(buf), 2, 4, C.addressof(buf), None)
        assert rc == Bn.ECUDA, L.cosenu_beam_sums_static_error()
