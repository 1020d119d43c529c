"""Rotation-sharded EMC iteration over several GPUs, one process per GPU (the paper's decomposition: PAPER.md:170,
188-194 Algorithm 2, 203; DESIGN.md section 11 NEXT-4).

Plumbing only: every rank holds the model, the detector, all patterns and the whole rotation list, works on its own
contiguous share of the rotations through the three libemc calls emc_shard_stats / emc_shard_update / emc_shard_finish,
and the two exchanges between them are torch.distributed collectives:

    all-gather   of the per-pattern statistics, 3 x ld_n floats per rank   (the paper: AllReduce(max) + AllReduce(sum) of
                 N floats; the statistics here are a reference pair + sum, merged in rank order on every rank)
    all-reduce   (sum) of the numerator and denominator grids, 2 n^3 floats (the paper: AllReduce of the model sums)

`backend` supplies the three phase functions (default: libemc through the binding); the CPU test of this module passes
an oracle-backed one, so that the sharding and the collectives are exercised without a GPU.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_bounds(n_rot: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous, balanced share [r0, r1) of `n_rot` rotations for `rank` of `world`."""
    return rank * n_rot // world, (rank + 1) * n_rot // world


class LibemcBackend:
    """The three device phases of a rank (include/emc.h, rotation shards)."""

    def __init__(self, flags=0):
        self.flags = flags
        self.ws = None

    def stats(self, model, q, mask, quat, weight, counts, n_rot_total):
        from . import binding as b

        st, self.ws = b.emc_shard_stats(model, q, mask, quat, weight, counts, n_rot_total, flags=self.flags, ws=self.ws)
        return st

    def update(self, model, q, mask, quat, weight, counts, n_rot_total, stats_all):
        from . import binding as b

        return b.emc_shard_update(model, q, mask, quat, weight, counts, n_rot_total, stats_all, self.ws, flags=self.flags)

    def finish(self, numden):
        from . import binding as b

        return b.emc_shard_finish(numden)


def _via_host(group) -> bool:
    """gloo moves CPU tensors: stage device tensors through the host for its collectives."""
    return dist.get_backend(group) == "gloo"


def all_gather_stats(stats: torch.Tensor, group=None) -> torch.Tensor:
    """[3, ld_n] per rank -> [world, 3, ld_n] in rank order (identical on every rank)."""
    world = dist.get_world_size(group)
    src = stats.cpu() if (stats.is_cuda and _via_host(group)) else stats
    parts = [torch.empty_like(src) for _ in range(world)]
    dist.all_gather(parts, src.contiguous(), group=group)
    return torch.stack(parts).to(stats.device)


def all_reduce_sum(x: torch.Tensor, group=None) -> torch.Tensor:
    if x.is_cuda and _via_host(group):
        h = x.cpu()
        dist.all_reduce(h, op=dist.ReduceOp.SUM, group=group)
        return h.to(x.device)
    dist.all_reduce(x, op=dist.ReduceOp.SUM, group=group)
    return x


def iterate_sharded(model, q, mask, quat, weight, counts, n_iter=1, group=None, backend=None, flags=0):
    """`n_iter` EMC iterations with the rotation list `quat` [R, 4] (and `weight` [R] or None) sharded over the ranks
    of `group` (default: the world).  Every rank passes the same arguments and gets the same results:
    dict(model, loglik [n_iter] float64, s = this rank's share of s[r], bounds = (r0, r1))."""
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    n_rot = quat.shape[0]
    r0, r1 = shard_bounds(n_rot, world, rank)
    if r1 <= r0:
        raise ValueError("fewer rotations than ranks")
    be = backend or LibemcBackend(flags)
    q_loc = quat[r0:r1].contiguous()
    w_loc = None if weight is None else weight[r0:r1].contiguous()
    ll, s = [], None
    for _ in range(n_iter):
        st = be.stats(model, q, mask, q_loc, w_loc, counts, n_rot)
        st_all = all_gather_stats(st, group)
        numden, ll_it, s = be.update(model, q, mask, q_loc, w_loc, counts, n_rot, st_all)
        numden = all_reduce_sum(numden, group)
        model = be.finish(numden)
        ll.append(ll_it.reshape(-1)[:1].double())
    return dict(model=model, loglik=torch.cat(ll), s=s, bounds=(r0, r1))
