"""Multi-GPU scale-out of the TSM loop: by source.

Sources are independent, so every rank holds a full gauge replica and runs the TSM loop on its own
share of ONE (N_LP, N_HP) workload: rank k of W takes the global sources r = k, k + W, k + 2W, ... (``shard``), which
spreads the first N_HP sources -- the ones that also get a high-precision solve -- evenly over the ranks.  The only
exchange is one all-reduce (sum) of the three raw momentum-space accumulators S_LP, S_LPc, S_HP
(3 x 160 * nmom * T complex128; 3 x 20 MB at 32^3x64) at the end; the division by N_LP and N_HP is done once, in the
library (``tsm_combine_sums``).  No collective exists inside the solver or the contraction, so there is nothing to
fuse with a compute kernel.  This module holds no TSM arithmetic: index bookkeeping and the collective only.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard(n_lp_total: int, n_hp_total: int, rank: int, world: int):
    """(n_lp_local, n_hp_local, src_first, src_stride) of rank `rank` of `world`: round-robin by global source index."""
    if not (0 <= rank < world):
        raise ValueError("shard: need 0 <= rank < world")
    if n_hp_total > n_lp_total:
        raise ValueError("shard: need n_hp_total <= n_lp_total")
    n_lp = len(range(rank, n_lp_total, world))
    n_hp = len(range(rank, n_hp_total, world))
    return n_lp, n_hp, rank, world


def allreduce_sums(sums: torch.Tensor, group=None) -> torch.Tensor:
    """In-place all-reduce (sum) of the raw accumulators [3, 2, 80, nmom, T] complex128 over the ranks."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        buf = torch.view_as_real(sums)          # complex all-reduce through the real view (nccl and gloo alike)
        dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
    return sums


def tsm_estimate_sharded(ctx, n_lp_total, n_hp_total, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, seed=0, z4=None,
                         group=None, **kw):
    """One (N_LP, N_HP) TSM workload split over the ranks of the process group: returns (estimate, info).

    z4 (optional): this rank's packed noise, [n_lp_local, 3V], local source j = global source rank + j * world."""
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    n_lp, n_hp, first, stride = shard(n_lp_total, n_hp_total, rank, world)
    shape = (3, 2, 80, len(momenta), ctx.T)
    if n_lp > 0:
        sums, _, info = ctx.tsm_estimate(n_lp, n_hp, kappa, mu, momenta, lp, hp, acc_lp, acc_hp, z4=z4, seed=seed,
                                         src_first=first, src_stride=stride, partial_sums=True, **kw)
    else:                                       # more ranks than sources: this rank contributes zeros
        sums, info = torch.zeros(shape, dtype=torch.complex128, device=ctx.tdev), {}
    allreduce_sums(sums, group)
    return ctx.tsm_combine_sums(sums, n_lp_total, n_hp_total), info
