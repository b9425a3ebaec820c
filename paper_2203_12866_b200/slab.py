"""z-slab decomposition drivers (include/cosenu.h "z-slab decomposition"; PAPER.md:341 names multi-GPU as future work).

The periodic z-grid is cut into contiguous slabs, one per GPU.  The velocity moments of Eq. (3) are local in z, so the
only exchange is the stencil halo (4 ghost rows per side), and that exchange is fused into the stage kernels: they store
their edge rows straight into the neighbouring slab's ghost rows over NVLink peer memory and bump an arrival counter there
(csrc/stage_kernels.cuh).  This module only moves handles and a few hundred bytes around:

* `slab_bounds`      -- the partition.
* `Ring`             -- neighbours of the periodic ring, exchange of peer descriptors, reduction of partials.
* `CosenuSlab`       -- one slab per process (one process per GPU, `torch.distributed` for the plumbing: the peer
                        descriptors are exchanged with all_gather_object, the diagnostics' partial sums with all_reduce).
* `SlabGroup`        -- several slabs driven by one process on one stream (used by the GPU tests to check the decomposed
                        path against the single-domain solver on one device).

No arithmetic of the method lives here: sums and maxima of the diagnostics' partials are the reduction the C ABI asks the
caller to supply.
"""
import ctypes as C

import numpy as np

from . import binding as B

NSUM, NMAX = 7, 3     # cosenu_slab_diag_sums: out[0..6] reduce by sum, out[7..9] by max


def slab_bounds(nz_global, world, rank):
    """Rows [z_begin, z_begin + nz_local) of slab `rank` of `world`: contiguous, remainder spread over the first slabs."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    base, rem = divmod(int(nz_global), int(world))
    if base < 16:
        raise ValueError("every slab needs at least 16 rows (nz_global=%d, world=%d)" % (nz_global, world))
    nz_local = base + (1 if rank < rem else 0)
    z_begin = rank * base + min(rank, rem)
    return z_begin, nz_local


def neighbours(world, rank):
    """(lo, hi) ranks of the periodic ring."""
    return (rank - 1) % world, (rank + 1) % world


def reduce_partials(parts):
    """Combine cosenu_slab_diag_sums arrays of several slabs: sums first, maxima last."""
    a = np.asarray(parts, dtype=np.float64).reshape(-1, NSUM + NMAX)
    return np.concatenate([a[:, :NSUM].sum(axis=0), a[:, NSUM:].max(axis=0)])


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _export(sim):
    peer = B.SlabPeer()
    sim._chk(sim._L.cosenu_slab_export(sim.h, C.byref(peer)))
    return peer


def _link(sim, lo, hi):
    sim._chk(sim._L.cosenu_slab_link(sim.h, C.byref(lo), C.byref(hi)))


def _ref_sums(sim):
    out = np.empty(4 * sim.nv, dtype=np.float64)
    sim._chk(sim._L.cosenu_slab_ref_sums(sim.h, _dp(out)))
    return out


def _diag_sums(sim):
    out = np.empty(NSUM + NMAX, dtype=np.float64)
    sim._chk(sim._L.cosenu_slab_diag_sums(sim.h, _dp(out)))
    return out


def _diag_finish(sim, g, set_reference):
    d = B.Diag()
    g = np.ascontiguousarray(g, dtype=np.float64)
    sim._chk(sim._L.cosenu_slab_diag_finish(sim.h, _dp(g), int(set_reference), C.byref(d)))
    return d.asdict()


def _wait_failed(sim):
    f = C.c_int32(0)
    sim._chk(sim._L.cosenu_slab_wait_failed(sim.h, C.byref(f)))
    return bool(f.value)


class Ring:
    """The `torch.distributed` plumbing of a decomposed run: who my neighbours are, exchange of the peer descriptors,
    reduction of the diagnostics' partials.  No device code: works under gloo on CPU (tests) and nccl alike."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self._dist = dist if (dist.is_available() and dist.is_initialized()) else None
        self._group = group
        self.world = self._dist.get_world_size(group) if self._dist else 1
        self.rank = self._dist.get_rank(group) if self._dist else 0
        self.lo, self.hi = neighbours(self.world, self.rank)

    def all_gather_bytes(self, blob):
        if not self._dist or self.world == 1:
            return [blob]
        out = [None] * self.world
        self._dist.all_gather_object(out, blob, group=self._group)
        return out

    def barrier(self):
        if self._dist and self.world > 1:
            self._dist.barrier(group=self._group)

    def all_reduce(self, arr, op):
        """arr: 1-D float64 numpy; op 'sum' or 'max' over the ranks (tiny arrays; device tensors under NCCL)."""
        if not self._dist or self.world == 1:
            return arr
        import torch
        dev = "cuda" if self._dist.get_backend(self._group) == "nccl" else "cpu"
        t = torch.from_numpy(np.ascontiguousarray(arr)).to(dev)
        self._dist.all_reduce(t, op=self._dist.ReduceOp.SUM if op == "sum" else self._dist.ReduceOp.MAX, group=self._group)
        return t.cpu().numpy()

    def reduce_diag_partials(self, p):
        """cosenu_slab_diag_sums of this rank -> the whole-grid array (sums first, maxima last)."""
        p = np.asarray(p, dtype=np.float64)
        return np.concatenate([self.all_reduce(p[:NSUM].copy(), "sum"), self.all_reduce(p[NSUM:].copy(), "max")])


class CosenuSlab:
    """This process's slab of a run decomposed over `torch.distributed` ranks (one process per GPU).

    With world == 1 (or torch.distributed not initialised) the slab is linked to itself: the single periodic domain,
    through the decomposed code path.
    """

    def __init__(self, nz_global, nv, L, dt, omega, theta, mu, scheme, group=None, **opts):
        self.ring = Ring(group)
        self.world, self.rank = self.ring.world, self.ring.rank
        self.nz_global, self.nv = int(nz_global), int(nv)
        self.z_begin, self.nz = slab_bounds(nz_global, self.world, self.rank)
        # the workspace is library-owned (cudaMalloc) so that its IPC handle names exactly this allocation
        import torch
        opts.setdefault("stream", torch.cuda.current_stream())
        self.sim = B.Cosenu(self.nz, nv, L, dt, omega, theta, mu, scheme, use_torch_workspace=False,
                            slab=(nz_global, self.z_begin), **opts)
        blobs = self.ring.all_gather_bytes(bytes(_export(self.sim)))
        _link(self.sim, B.SlabPeer.from_buffer_copy(blobs[self.ring.lo]), B.SlabPeer.from_buffer_copy(blobs[self.ring.hi]))
        self.ring.barrier()

    def _after_upload(self):
        self.sim._chk(self.sim._L.cosenu_slab_push_ghosts(self.sim.h))
        self.ring.barrier()                               # every slab's ghost rows are in place
        g = self.ring.all_reduce(_ref_sums(self.sim), "sum")
        self.sim._chk(self.sim._L.cosenu_slab_set_ref_sums(self.sim.h, _dp(np.ascontiguousarray(g))))
        _diag_finish(self.sim, self.ring.reduce_diag_partials(_diag_sums(self.sim)), True)

    # ---- the calls of the C ABI, on this rank's rows
    def init(self, seed, **kw):
        self.sim.init(seed, **kw)
        self._after_upload()

    def set_state(self, local_state, t=0.0):
        """local_state: (8, nz_local, nv) = rows [z_begin, z_begin + nz_local) of the global state."""
        self.sim.set_state(local_state, t)
        self._after_upload()

    def step(self, n=1):
        self.sim.step(n)

    def step_lockstep(self, n=1):
        """n steps with a device sync and a barrier over the ranks after EVERY stage: every arrival counter has reached its
        value before the next launch, so no kernel ever waits for another process.  This is how ranks that share one GPU
        must be driven (their kernels are time-sliced, not concurrent); with one GPU per rank use step()."""
        for _ in range(int(n)):
            for k in range(4):
                self.sim._chk(self.sim._L.cosenu_slab_stage(self.sim.h, k))
                self.sim.sync()
                self.ring.barrier()

    def sync(self):
        self.sim.sync()        # raises if a halo wait of this slab gave up (cosenu_sync checks the flag)

    def wait_failed(self):
        return _wait_failed(self.sim)

    def get_state(self, out=None):
        return self.sim.get_state(out)

    def get_moments(self):
        return self.sim.get_moments()

    def diagnostics(self):
        """Collective: every rank must call it."""
        return _diag_finish(self.sim, self.ring.reduce_diag_partials(_diag_sums(self.sim)), False)

    def launch_count(self):
        return self.sim.launch_count()

    def close(self):
        if self.sim is not None:
            self.sim.sync()
            self.ring.barrier()                           # nobody may still be writing into my ghost rows
            self.sim.close()
            self.sim = None


class SlabGroup:
    """`nslabs` slabs of one periodic grid in ONE process on ONE stream of the current device.

    The stage launches are issued stage by stage over all slabs (cosenu_slab_step_group), so no kernel ever waits for
    one queued behind it.  Same results as `Cosenu` on the whole grid, bit for bit (the per-cell arithmetic and the
    moment summation order do not depend on the decomposition).
    """

    def __init__(self, nslabs, nz_global, nv, L, dt, omega, theta, mu, scheme, bounds=None, **opts):
        import torch
        self.nz_global, self.nv = int(nz_global), int(nv)
        self.bounds = bounds if bounds is not None else [slab_bounds(nz_global, nslabs, r) for r in range(nslabs)]
        # one real (capturable, non-legacy) stream for the whole group: a NULL stream would make every handle create its own
        self._stream = st = torch.cuda.Stream()
        self.sims = [B.Cosenu(nzl, nv, L, dt, omega, theta, mu, scheme, use_torch_workspace=False, stream=st,
                              slab=(nz_global, zb), **opts) for zb, nzl in self.bounds]
        peers = [_export(s) for s in self.sims]
        n = len(self.sims)
        for r, s in enumerate(self.sims):
            lo, hi = neighbours(n, r)
            _link(s, peers[lo], peers[hi])
        self._L = self.sims[0]._L
        self._arr = (C.c_void_p * n)(*[s.h for s in self.sims])

    def _after_upload(self):
        for s in self.sims:
            s._chk(self._L.cosenu_slab_push_ghosts(s.h))
        g = np.sum([_ref_sums(s) for s in self.sims], axis=0)
        for s in self.sims:
            s._chk(self._L.cosenu_slab_set_ref_sums(s.h, _dp(np.ascontiguousarray(g))))
        g = reduce_partials([_diag_sums(s) for s in self.sims])
        for s in self.sims:
            _diag_finish(s, g, True)

    def init(self, seed, **kw):
        for s in self.sims:
            s.init(seed, **kw)
        self._after_upload()

    def set_state(self, state, t=0.0):
        assert state.shape == (8, self.nz_global, self.nv)
        for s, (zb, nzl) in zip(self.sims, self.bounds):
            s.set_state(np.ascontiguousarray(state[:, zb:zb + nzl, :]), t)
        self._after_upload()

    def step(self, n=1):
        rc = self._L.cosenu_slab_step_group(self._arr, len(self.sims), n)
        if rc != 0:
            msgs = [self._L.cosenu_last_error(s.h).decode() for s in self.sims]
            raise B.CosenuError(rc, "; ".join(m for m in msgs if m))

    def sync(self):
        for s in self.sims:
            s.sync()           # raises if a halo wait of that slab gave up

    def get_state(self):
        return np.concatenate([s.get_state() for s in self.sims], axis=1)

    def get_moments(self):
        return np.concatenate([s.get_moments() for s in self.sims], axis=1)

    def diagnostics(self):
        g = reduce_partials([_diag_sums(s) for s in self.sims])
        return _diag_finish(self.sims[0], g, False)

    def launch_count(self):
        return sum(s.launch_count() for s in self.sims)

    def close(self):
        for s in self.sims:
            s.sync()
        for s in self.sims:
            s.close()
        self.sims = []


class ConcurrentSlabs(SlabGroup):
    """`nslabs` slabs of one periodic grid in ONE process on ONE device, every slab on a stream of its OWN and driven by a host
    thread of its own with the free-running `cosenu_step(n)`: no host synchronisation between the stages, nothing orders the
    slabs' launches but the arrival counters in device memory.  With `max_ctas` <= (SMs / nslabs) the stage kernels of all
    slabs are co-resident (one CTA per SM each), so the kernels really spin on each other: this is the halo-exchange
    protocol of a multi-GPU run (RAW wait, WAR argument of DESIGN.md section 8) on one GPU.
    """

    def __init__(self, nslabs, nz_global, nv, L, dt, omega, theta, mu, scheme, max_ctas, bounds=None,
                 blocking_streams=False, **opts):
        """blocking_streams: every handle creates its own plain cudaStreamCreate stream (one that synchronises with the
        legacy default stream) instead of using a non-blocking torch stream."""
        import torch
        self.nz_global, self.nv = int(nz_global), int(nv)
        self.bounds = bounds if bounds is not None else [slab_bounds(nz_global, nslabs, r) for r in range(nslabs)]
        self._streams = [None if blocking_streams else torch.cuda.Stream() for _ in self.bounds]
        self.sims = [B.Cosenu(nzl, nv, L, dt, omega, theta, mu, scheme, use_torch_workspace=False, stream=st,
                              slab=(nz_global, zb), **opts) for (zb, nzl), st in zip(self.bounds, self._streams)]
        for s in self.sims:
            s.set_option(B.OPT_MAX_CTAS, max_ctas)
        peers = [_export(s) for s in self.sims]
        n = len(self.sims)
        for r, s in enumerate(self.sims):
            lo, hi = neighbours(n, r)
            _link(s, peers[lo], peers[hi])
        self._L = self.sims[0]._L

    def step(self, n=1, delays=None, sync_every_step=None):
        """Every slab's thread enqueues its n steps (4 n launches) on its own stream; delays[r] seconds of head start skew.
        sync_every_step[r]: that slab's thread runs step(1) + sync n times instead (a driver that looks at every step)."""
        import threading
        import time
        errs = [None] * len(self.sims)

        def run(r):
            try:
                if delays and delays[r]:
                    time.sleep(delays[r])
                if sync_every_step and sync_every_step[r]:
                    for _ in range(n):
                        self.sims[r].step(1)
                        self.sims[r].sync()
                else:
                    self.sims[r].step(n)
            except Exception as e:   # noqa: BLE001  (reported to the caller below)
                errs[r] = e

        th = [threading.Thread(target=run, args=(r,)) for r in range(len(self.sims))]
        for t in th:
            t.start()
        for t in th:
            t.join()
        for e in errs:
            if e is not None:
                raise e
