"""Multi-GPU drivers: one process per GPU, torch.distributed for the plumbing.

LORs / events are independent units: every rank holds a contiguous shard of the list and the whole image (15 MB).
Forward projections need no exchange (outputs are disjoint); a back projection, and every OSEM subset update, needs
ONE all-reduce(sum) of the image -- the device-side form of the paper's host-staged multi-GPU fan-out.  This module
holds only that plumbing (sharding rules, the order of calls and the collective); all arithmetic is in the C-ABI
calls passed in as ``ops`` (on a GPU: ``CudaOps``, i.e. libjoseph_b200 through ``binding``).  The CPU tests drive
the same functions over ``gloo`` with an ``ops`` of their own.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_events(n: int, rank: int, world: int, n_subsets: int = 1):
    """Contiguous [lo, hi) shard of ``n`` events whose start is a multiple of ``n_subsets`` (so that the subset of a
    local event, local index mod n_subsets, is the subset of the global event) and of 32."""
    import math
    align = n_subsets * 32 // math.gcd(n_subsets, 32)
    per = -(-n // world)
    per = -(-per // align) * align
    lo = min(n, rank * per)
    return lo, min(n, lo + per)


def _all_reduce_sum(t: torch.Tensor, group=None):
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t


def back_sharded(ops, y_local, img_out: torch.Tensor, group=None) -> torch.Tensor:
    """img_out = sum over ranks of A_shard^T y_shard (img_out is overwritten on every rank with the full result)"""
    img_out.zero_()
    ops.back(y_local, img_out)
    return _all_reduce_sum(img_out, group)


def lm_osem_sharded(ops, sens: torch.Tensor, x: torch.Tensor, n_subsets: int, n_iter: int, group=None) -> torch.Tensor:
    """Listmode OSEM (reading A14) over event shards: per subset every rank computes b = A_m^T (1 / (A_m x)) over its
    own events (``ops.backratio``), the images b are summed over the ranks, and every rank applies the same update
    x <- x b n_subsets / sens (``ops.update``), so x stays replicated.  ``sens`` is the global sensitivity image."""
    b = torch.empty_like(x)
    for _ in range(int(n_iter)):
        for m in range(int(n_subsets)):
            ops.backratio(m, x, b)
            _all_reduce_sum(b, group)
            ops.update(x, b, sens, float(n_subsets))
    return x


class CudaOps:
    """The C-ABI calls behind the drivers above, bound to this rank's shard (a listmode plan and / or a LOR list)."""

    def __init__(self, jp, plan=None, lors=None, geom=None):
        self.jp, self.plan, self.lors, self.geom = jp, plan, lors, geom
        self.ws = None

    def back(self, y_local, img):
        xs, xe = self.lors
        g = self.geom
        self.jp.jp_back(xs, xe, y_local, g.n, g.origin, g.voxsize, img=img)

    def backratio(self, subset, x, b):
        if self.ws is None:
            need = int(self.jp.load().jp_lm_osem_planned_workspace_bytes(self.plan.handle))
            self.ws = torch.empty(need, dtype=torch.uint8, device=x.device)
        self.jp.jp_lm_osem_planned_backratio(self.plan, subset, x, out=b, workspace=self.ws)

    def update(self, x, b, sens, scale):
        self.jp.jp_osem_update(x, b, sens, scale)
