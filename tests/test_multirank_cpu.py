"""The N > 1 plumbing of bench.py on CPU: world_size-2 gloo, max-over-ranks timing and whole-job aggregation;
the reference arm runs on rank 0 only."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, device="cpu")          # slowest rank decides
    value = bench.whole_job_value(cells=1000, steps=4, world=world, ms=ms)
    dist.barrier()
    q.put((rank, ms, value))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo():
    from conftest import free_port
    port = free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert [o[1] for o in out] == [15.0, 15.0]
    assert all(abs(o[2] - 2 * 1000 * 4 / 15e-3) < 1e-6 for o in out)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_reference_arm_json_line():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg0",
                        "--steps", "2", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["unit"] == "cell-updates/s"


# ---------------------------------------------------------------------------------------------------------
# z-slab decomposition plumbing (paper_2203_12866_b200/slab.py) on CPU: partition, ring neighbours, exchange of the
# peer descriptors as bytes, reduction of the diagnostics' partial arrays (sums first, maxima last).
def test_slab_bounds_cover_the_grid():
    from paper_2203_12866_b200 import slab
    for nz, world in ((1024, 1), (1024, 2), (1000, 3), (262144, 8), (131, 8), (16 * 5 + 3, 5)):
        b = [slab.slab_bounds(nz, world, r) for r in range(world)]
        assert b[0][0] == 0 and sum(n for _, n in b) == nz
        for (z0, n0), (z1, _) in zip(b, b[1:]):
            assert z0 + n0 == z1
        assert max(n for _, n in b) - min(n for _, n in b) <= 1 and min(n for _, n in b) >= 16
    import pytest
    with pytest.raises(ValueError):
        slab.slab_bounds(100, 8, 0)      # slabs thinner than a tile
    assert slab.neighbours(4, 0) == (3, 1) and slab.neighbours(1, 0) == (0, 0) and slab.neighbours(2, 1) == (0, 0)


def _slab_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import ctypes
    import numpy as np
    from paper_2203_12866_b200 import binding as B, slab
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ring = slab.Ring()
    # a peer descriptor as the library would fill it, sent as bytes
    me = B.SlabPeer()
    me.pid, me.nz_local, me.off_ctr, me.nvp = 1000 + rank, 64 + rank, 4096 * (rank + 1), 16
    for k in range(64):
        me.ipc_handle[k] = (rank * 64 + k) % 256
    blobs = ring.all_gather_bytes(bytes(me))
    lo, hi = B.SlabPeer.from_buffer_copy(blobs[ring.lo]), B.SlabPeer.from_buffer_copy(blobs[ring.hi])
    part = np.arange(10, dtype=np.float64) * (rank + 1)          # sums [0..6], maxima [7..9]
    red = ring.reduce_diag_partials(part)
    ring.barrier()
    q.put((rank, ring.lo, ring.hi, int(lo.pid), int(hi.nz_local), int(lo.ipc_handle[5]), len(blobs[0]),
           ctypes.sizeof(B.SlabPeer), red.tolist()))
    dist.destroy_process_group()


def test_slab_ring_plumbing_gloo():
    import numpy as np
    from conftest import free_port
    port = free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    world = 2
    ps = [ctx.Process(target=_slab_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, lo, hi, lo_pid, hi_nz, lo_byte, blob_len, size, red in out:
        assert (lo, hi) == ((rank - 1) % world, (rank + 1) % world)
        assert lo_pid == 1000 + lo and hi_nz == 64 + hi and lo_byte == (lo * 64 + 5) % 256
        assert blob_len == size
        base = np.arange(10, dtype=np.float64)
        assert red[:7] == (base[:7] * 3).tolist()               # 1x + 2x summed
        assert red[7:] == (base[7:] * 2).tolist()               # max over ranks
