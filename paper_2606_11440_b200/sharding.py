"""Env-sharded multi-GPU runs: host-side logic only, no data-path collective.

Environments are independent and every random draw is keyed by the GLOBAL env id (R2), so rank r of W simply owns a
contiguous range of env ids; its result is bit-identical to the same columns of a single-GPU run.  The one collective of
a training step is the all-reduce of the four sums behind C-bar and the utility normalisation
(PAPER.md:127-129): sum of costs, number of finalised queries, sum U, sum U^2.
"""
from __future__ import annotations

import math
from typing import Dict, Tuple


def shard_range(n_envs_total: int, rank: int, world: int) -> Tuple[int, int]:
    """(first env, count) of rank `rank`: contiguous ranges, the remainder spread over the first ranks."""
    if not (0 <= rank < world) or n_envs_total < world:
        raise ValueError("need 0 <= rank < world <= n_envs_total")
    q, r = divmod(n_envs_total, world)
    return rank * q + min(rank, r), q + (1 if rank < r else 0)


def shard_spec(spec, rank: int, world: int):
    """PoolSpec of one rank of a STRONG-scaling split of `spec` (same global env ids as the unsharded run)."""
    base, cnt = shard_range(spec.n_envs, rank, world)
    scale = lambda cap: max(1024, int(cap) * cnt // spec.n_envs + 1024)
    return spec.with_(n_envs=cnt, env_id_base=int(spec.env_id_base) + base, env_level=spec.env_level[base:base + cnt].copy(),
                      log_cap_exec=scale(spec.log_cap_exec), log_cap_plan=scale(spec.log_cap_plan), log_cap_query=scale(spec.log_cap_query))


def partial_sums(scalars: Dict[str, float]) -> Tuple[float, float, float, float]:
    """(sum_cost, n_final, sum_U, sum_U2) of one rank from its SCALARS telemetry."""
    n = float(scalars["n_final"])
    return (float(scalars["sum_cost"]), n, float(scalars["ubar"]) * n, (float(scalars["usigma"]) ** 2 + float(scalars["ubar"]) ** 2) * n)


def combine_sums(sum_cost: float, n_final: float, sum_u: float, sum_u2: float) -> Dict[str, float]:
    """C-bar, U-bar, sigma_U of the whole job from the reduced sums (R32: population std)."""
    if n_final <= 0:
        return dict(cbar=0.0, ubar=0.0, usigma=0.0, sum_cost=sum_cost, n_final=0)
    ubar = sum_u / n_final
    var = max(sum_u2 / n_final - ubar * ubar, 0.0)
    return dict(cbar=sum_cost / n_final, ubar=ubar, usigma=math.sqrt(var), sum_cost=sum_cost, n_final=int(round(n_final)))


def allreduce_scalars(scalars: Dict[str, float], device="cpu", group=None) -> Dict[str, float]:
    """The step's one collective: SUM all-reduce of the four sums over the process group (NCCL on GPUs, gloo in tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(partial_sums(scalars), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return combine_sums(*[float(x) for x in t.tolist()])
