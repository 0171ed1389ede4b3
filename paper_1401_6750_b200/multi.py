"""Multi-GPU scale-out of the TSM loop: by source.

Sources are independent, so every rank holds a full gauge replica, runs
``tsm_estimate`` on its own block of sources and the only exchange is one all-reduce of the
momentum-space estimate (160 * nmom * T complex128; 20 MB at 32^3x64) at the end.  No data-path
collective exists inside the solver or the contraction.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def rank_seed(seed: int, rank: int) -> int:
    """Noise seed of a rank: disjoint counter-hash streams per rank."""
    return int(seed) + 1000003 * int(rank)


def combine_over_ranks(local_estimate: torch.Tensor, n_lp_local: int, n_hp_local: int, group=None) -> torch.Tensor:
    """Global TSM estimate from per-rank estimates.

    L = sum_ranks (n_lp_r / N_LP) L_r, valid when every rank has the same N_HP/N_LP ratio (then
    the LP mean and the correction mean are both weighted by n_lp_r / N_LP); checked here."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return local_estimate
    counts = torch.tensor([float(n_lp_local), float(n_hp_local)], dtype=torch.float64, device=local_estimate.device)
    allc = [torch.empty_like(counts) for _ in range(dist.get_world_size(group))]
    dist.all_gather(allc, counts, group=group)
    n_lp = sum(float(c[0]) for c in allc)
    n_hp = sum(float(c[1]) for c in allc)
    for c in allc:
        if abs(float(c[1]) * n_lp - float(c[0]) * n_hp) > 1e-9 * max(1.0, n_lp * n_hp):
            raise ValueError("combine_over_ranks: ranks must share the same N_HP / N_LP ratio")
    # complex all-reduce through the real view (works for nccl and gloo alike)
    buf = torch.view_as_real(local_estimate * (n_lp_local / n_lp)).contiguous()
    dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
    return torch.view_as_complex(buf)
