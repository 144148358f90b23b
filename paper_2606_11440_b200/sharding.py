"""Env-sharded multi-GPU runs: host-side logic only, no data-path collective.

Environments are independent and every random draw is keyed by the GLOBAL env id (R2), so rank r of W simply owns a
contiguous range of env ids; its trajectories are bit-identical to the same columns of a single-GPU run.  The one
collective of a training step is the SUM all-reduce of the four sums behind C-bar and the utility
normalisation: sum of costs, number of finalised queries, sum U, sum U^2 (IM_TEL_SUMS).  The
arithmetic on those sums lives in the library (im_returns_finish); nothing here computes.
"""
from __future__ import annotations

from typing import Tuple

import numpy as np


def shard_range(n_envs_total: int, rank: int, world: int) -> Tuple[int, int]:
    """(first env, count) of rank `rank`: contiguous ranges, the remainder spread over the first ranks."""
    if not (0 <= rank < world) or n_envs_total < world:
        raise ValueError("need 0 <= rank < world <= n_envs_total")
    q, r = divmod(n_envs_total, world)
    return rank * q + min(rank, r), q + (1 if rank < r else 0)


def shard_spec(spec, rank: int, world: int):
    """PoolSpec of one rank of a STRONG-scaling split of `spec` (same global env ids as the unsharded run).

    Log capacities are sized from the shard's OWN arrival levels (contiguous shards of a utilisation sweep differ a
    lot in load); a capacity of 0 ("library default") is passed through."""
    base, cnt = shard_range(spec.n_envs, rank, world)
    lv = np.asarray(spec.env_level[base:base + cnt], dtype=np.int64)
    rate = np.asarray(spec.arr_rate_tick, dtype=np.float64)
    whole = float(rate[np.asarray(spec.env_level, dtype=np.int64)].sum()) if len(rate) else 0.0
    share = float(rate[lv].sum()) / whole if whole > 0 else cnt / spec.n_envs
    scale = lambda cap: 0 if int(cap) == 0 else int(int(cap) * share * 1.25) + 64 * cnt + 4096
    return spec.with_(n_envs=cnt, env_id_base=int(spec.env_id_base) + base, env_level=spec.env_level[base:base + cnt].copy(),
                      log_cap_exec=scale(spec.log_cap_exec), log_cap_plan=scale(spec.log_cap_plan), log_cap_query=scale(spec.log_cap_query))


def allreduce_sums(sums, device="cpu", group=None) -> np.ndarray:
    """The step's one collective: SUM all-reduce of [sum_cost, n_final, sum_U, sum_U2] over the process group
    (NCCL on GPUs, gloo in tests).  Returns the job-wide sums as a float64 numpy array for im_returns_finish."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(np.asarray(sums, dtype=np.float64), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t.cpu().numpy()
