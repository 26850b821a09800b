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


# ---- listmode OSEM over event shards (multi_gpu.lm_osem_sharded): one all-reduce of the image per subset --------
TOF_LM = (9.0, 7.0, 3.0)


class _OracleOps:
    """per-shard arithmetic of the drivers in multi_gpu.py done by the oracle (CPU, float64)"""

    def __init__(self, xs, xe, tb, geom, n_subsets):
        self.xs, self.xe, self.tb, self.g, self.ns = xs, xe, tb, geom, n_subsets

    def backratio(self, m, x, b):
        import oracle
        sl = slice(m, None, self.ns)
        xs, xe, tb = self.xs[:, sl], self.xe[:, sl], self.tb[sl]
        out = np.zeros(self.g.n)
        if xs.shape[1]:
            p = oracle.fwd_tof_lm(xs, xe, tb, x.numpy(), self.g.origin, self.g.voxsize, *TOF_LM)
            r = np.where(p > 1e-9, 1.0 / np.where(p > 1e-9, p, 1.0), 0.0)
            out = oracle.back_tof_lm(xs, xe, tb, r, self.g.n, self.g.origin, self.g.voxsize, *TOF_LM)
        b.copy_(torch.from_numpy(out))

    def update(self, x, b, sens, scale):
        x.copy_(torch.where(sens > 0, x * b * scale / torch.where(sens > 0, sens, torch.ones_like(sens)),
                            torch.zeros_like(x)))
        b.zero_()


def _osem_worker(rank, world, port, n_ev, n_subsets, q):
    from paper_2212_12519_b200 import multi_gpu
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = inputs.config0(n_lors=n_ev)
    g = c["geom"]
    tb = np.random.default_rng(7).integers(-4, 5, n_ev).astype(np.int16)
    lo, hi = multi_gpu.shard_events(n_ev, rank, world, n_subsets)
    ops = _OracleOps(c["xstart"][:, lo:hi], c["xend"][:, lo:hi], tb[lo:hi], g, n_subsets)
    sens = torch.ones(g.n, dtype=torch.float64)
    x = torch.ones(g.n, dtype=torch.float64)
    multi_gpu.lm_osem_sharded(ops, sens, x, n_subsets, 2)
    if rank == 0:
        q.put(x.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_shard_events_keeps_subsets():
    from paper_2212_12519_b200 import multi_gpu
    for n in (0, 5, 1000, 40_000_000):
        for world in (1, 2, 3, 8):
            for ns in (1, 3, 20):
                spans = [multi_gpu.shard_events(n, r, world, ns) for r in range(world)]
                assert spans[0][0] == 0 and spans[-1][1] == n
                assert all(a1 == b0 for (_, a1), (b0, _) in zip(spans[:-1], spans[1:]))
                assert all(lo % ns == 0 or lo == n for lo, _ in spans)


def test_world2_gloo_sharded_osem():
    import oracle
    n_ev, world, n_subsets = 2500, 2, 3
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_osem_worker, args=(r, world, port, n_ev, n_subsets, q)) for r in range(world)]
    for p in procs:
        p.start()
    x = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    c = inputs.config0(n_lors=n_ev)
    g = c["geom"]
    tb = np.random.default_rng(7).integers(-4, 5, n_ev).astype(np.int16)
    ref = oracle.lm_osem(c["xstart"], c["xend"], tb, np.ones(g.n), np.ones(g.n), g.origin, g.voxsize, *TOF_LM,
                         n_subsets=n_subsets, n_iter=2)
    assert np.abs(x - ref).max() <= 1e-12 * np.abs(ref).max()
