"""Guard bands in place of compute-sanitizer (closed on this pool; SURVEY.md section 5 "race detection / sanitizers").

The stage kernels move almost everything with TMA, which clips at the tensor's edges, but three kinds of store are issued
thread by thread with computed addresses: the ghost rows of a stage output (own buffer or, for slabs, the NEIGHBOUR's
workspace), the moments, and the arrival counters.  Here every workspace is carved out of a larger torch buffer with 1 MiB
of a NaN-free bit pattern on both sides; after runs on ragged, tiny and decomposed shapes every guard byte must be
untouched.  Slabs are given adjacent carve-outs of ONE buffer, so a store that overshoots a neighbour's ghost rows lands in a
guard band (or in the next slab's workspace, where the bitwise comparison with the single domain catches it).
Also checked: the row-pitch padding columns (nvp > nv) of the state buffers stay exactly zero (the zero fill of the
workspace is all that ever writes them)."""
import ctypes as C

import numpy as np
import pytest

from paper_2203_12866_b200 import inputs

pytestmark = pytest.mark.gpu

FD, FV = 0, 1
GUARD = 1 << 20
PATTERN = 0xA5


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2203_12866_b200 import binding
    binding.load()
    return binding


class Arena:
    """One torch buffer: guard | workspace 0 | guard | workspace 1 | guard ..., every guard byte = PATTERN."""

    def __init__(self, sizes):
        import torch
        self.sizes = [(int(n) + 255) // 256 * 256 for n in sizes]
        total = GUARD + sum(n + GUARD for n in self.sizes)
        self.buf = torch.full((total,), PATTERN, dtype=torch.uint8, device="cuda")
        self.offs, o = [], GUARD
        for n in self.sizes:
            self.offs.append(o)
            o += n + GUARD
        assert self.buf.data_ptr() % 256 == 0

    def ptr(self, k):
        return self.buf.data_ptr() + self.offs[k]

    def assert_guards_untouched(self):
        import torch
        torch.cuda.synchronize()
        lo = 0
        for o, n in zip(self.offs, self.sizes):
            g = self.buf[lo:o]
            assert bool((g == PATTERN).all()), "guard band before the workspace at byte %d was written" % o
            lo = o + n
        assert bool((self.buf[lo:] == PATTERN).all()), "guard band after the last workspace was written"


def test_the_guard_check_sees_a_single_stray_byte(B):
    arena = Arena([4096, 8192])
    arena.assert_guards_untouched()
    arena.buf[arena.offs[1] - 1] = 0          # last byte of the guard between the two workspaces
    with pytest.raises(AssertionError):
        arena.assert_guards_untouched()


def _attach(B, sim, arena, k, stream):
    L = B.load()
    need = L.cosenu_workspace_bytes(sim.h)
    assert need <= arena.sizes[k]
    sim._chk(L.cosenu_attach(sim.h, C.c_void_p(arena.ptr(k)), need, stream.cuda_stream))


def _need(B, args, slab=None):
    s = B.Cosenu(*args, use_torch_workspace=False, slab=slab)
    n = s.workspace_bytes()
    s.close()
    return n


SHAPES = [(16, 2), (17, 3), (50, 33), (200, 20), (250, 100), (333, 130), (1024, 16), (4096, 64)]   # tiny, ragged, cfg0, cfg1


@pytest.mark.parametrize("scheme", [FD, FV])
@pytest.mark.parametrize("nz,nv", SHAPES)
def test_single_domain_stays_inside_its_workspace(B, scheme, nz, nv):
    import torch
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
    arena = Arena([_need(B, args)])
    st = inputs.random_state(nz, nv, seed=5000 + nz + nv)
    ref = B.Cosenu(*args)
    ref.set_state(st)
    ref.step(6)
    want = ref.get_state()
    ref.close()
    stream = torch.cuda.Stream()
    sim = B.Cosenu(*args, use_torch_workspace=False)
    _attach(B, sim, arena, 0, stream)
    sim.set_state(st)
    sim.step(6)
    sim.diagnostics()
    got = sim.get_state()
    sim.close()
    assert np.array_equal(got, want)
    arena.assert_guards_untouched()


@pytest.mark.parametrize("scheme", [FD, FV])
@pytest.mark.parametrize("nz,nv,nslabs", [(64, 5, 2), (250, 100, 3), (333, 130, 2), (1024, 16, 4)])
def test_slabs_stay_inside_their_workspaces(B, scheme, nz, nv, nslabs):
    """Neighbouring slabs in adjacent carve-outs: the peer stores into ghost rows and the counter updates stay inside the
    neighbour's workspace (guards intact) and hit the right rows (bitwise the single domain)."""
    import torch
    from paper_2203_12866_b200 import slab as S
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
    st = inputs.random_state(nz, nv, seed=6000 + nz + nv)
    ref = B.Cosenu(*args)
    ref.set_state(st)
    ref.step(5)
    want, wantm = ref.get_state(), ref.get_moments()
    ref.close()
    bounds = [S.slab_bounds(nz, nslabs, r) for r in range(nslabs)]
    tail = args[2:]
    arena = Arena([_need(B, (nzl, nv) + tail, slab=(nz, zb)) for zb, nzl in bounds])
    stream = torch.cuda.Stream()
    grp = S.SlabGroup.__new__(S.SlabGroup)          # SlabGroup's driver logic on workspaces of our own
    grp.nz_global, grp.nv, grp.bounds, grp._stream = nz, nv, bounds, stream
    grp.sims = []
    for k, (zb, nzl) in enumerate(bounds):
        s = B.Cosenu(nzl, nv, *tail, use_torch_workspace=False, slab=(nz, zb))
        _attach(B, s, arena, k, stream)
        grp.sims.append(s)
    peers = [S._export(s) for s in grp.sims]
    for r, s in enumerate(grp.sims):
        lo, hi = S.neighbours(nslabs, r)
        S._link(s, peers[lo], peers[hi])
    grp._L = grp.sims[0]._L
    grp._arr = (C.c_void_p * nslabs)(*[s.h for s in grp.sims])
    grp.set_state(st)
    grp.step(5)
    grp.sync()
    grp.diagnostics()
    got, gotm = grp.get_state(), grp.get_moments()
    grp.close()
    assert np.array_equal(got, want)
    assert np.array_equal(gotm, wantm)
    arena.assert_guards_untouched()


@pytest.mark.parametrize("scheme", [FD, FV])
def test_row_pitch_padding_stays_zero(B, scheme):
    """nv = 33 is padded to a longer row pitch: the padding columns of all four state buffers are never written."""
    import torch
    nz, nv = 100, 33
    args = (nz, nv, 0.7 * nz, 0.05, 0.8, 0.3, 1.3, scheme)
    arena = Arena([_need(B, args)])
    stream = torch.cuda.Stream()
    sim = B.Cosenu(*args, use_torch_workspace=False)
    _attach(B, sim, arena, 0, stream)
    sim.set_state(inputs.random_state(nz, nv, seed=7))
    sim.step(4)
    sim.sync()
    # layout (csrc/cosenu_api.cu workspace_layout): four state buffers [8][nz + 2 G][nvp] doubles at the start of the workspace,
    # nvp = nv rounded up to a multiple of 4 (32-byte rows), each buffer rounded up to 256 bytes; U is the first
    G, nvp = 4, (nv + 3) // 4 * 4
    assert nvp > nv
    rows = 8 * (nz + 2 * G)
    st_elems = (rows * nvp * 8 + 255) // 256 * 256 // 8
    ws = arena.buf[arena.offs[0]:arena.offs[0] + arena.sizes[0]].view(torch.float64)
    sim.close()
    bufs = [ws[b * st_elems:b * st_elems + rows * nvp].view(rows, nvp) for b in range(4)]
    assert bool((bufs[0][:, :nv] != 0).any())                     # the layout assumption: U's data columns hold the state
    for b, x in enumerate(bufs):
        assert bool((x[:, nv:] == 0).all()), "padding columns of state buffer %d were written" % b
    arena.assert_guards_untouched()
