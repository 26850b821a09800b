"""Multi-GPU host logic on CPU: world_size-2 gloo.  LORs are independent units: each
rank takes a contiguous shard, forward outputs are disjoint, the back-projected image is the
all-reduce(sum) of the per-shard images.  No GPU here, so the per-shard arithmetic is done by the
oracle -- what is under test is the sharding / reduction plumbing that bench.py and a multi-GPU
caller use (inputs.shard_range + torch.distributed)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2212_12519_b200 import inputs


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_lors, q):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = inputs.config0(n_lors=n_lors)
    g = c["geom"]
    lo, hi = inputs.shard_range(n_lors, rank, world)
    xs, xe = c["xstart"][:, lo:hi], c["xend"][:, lo:hi]
    p = oracle.fwd(xs, xe, c["img"], g.origin, g.voxsize)
    b = torch.from_numpy(oracle.back(xs, xe, c["y"][lo:hi], g.n, g.origin, g.voxsize))
    dist.all_reduce(b, op=dist.ReduceOp.SUM)                      # the one exchange step of the adjoint
    counts = torch.tensor([hi - lo], dtype=torch.int64)
    dist.all_reduce(counts)
    t = torch.tensor([1.0 + rank], dtype=torch.float64)           # "max over ranks" timing reduction
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    gathered = [None] * world
    dist.all_gather_object(gathered, (lo, hi, p))
    if rank == 0:
        q.put((b.numpy(), int(counts[0]), float(t[0]), gathered))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_range_partitions():
    for n in (0, 1, 31, 32, 33, 50_000, 151_584_768):
        for world in (1, 2, 3, 8):
            spans = [inputs.shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for (a0, a1), (b0, b1) in zip(spans[:-1], spans[1:]):
                assert a1 == b0 and a0 <= a1
            assert all(lo % 32 == 0 or lo == n for lo, _ in spans)


def test_world2_gloo_sharded_projection():
    import oracle
    n_lors, world = 3001, 2
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_lors, q)) for r in range(world)]
    for p in procs:
        p.start()
    b, count, tmax, gathered = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert count == n_lors and tmax == 2.0
    c = inputs.config0(n_lors=n_lors)
    g = c["geom"]
    ref_b = oracle.back(c["xstart"], c["xend"], c["y"], g.n, g.origin, g.voxsize)
    assert np.allclose(b, ref_b, rtol=1e-12, atol=1e-12)
    ref_p = oracle.fwd(c["xstart"], c["xend"], c["img"], g.origin, g.voxsize)
    full = np.empty(n_lors)
    for lo, hi, p in gathered:
        full[lo:hi] = p
    assert np.array_equal(full, ref_p)
