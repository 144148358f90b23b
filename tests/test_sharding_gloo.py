"""N > 1 path on CPU: world_size 2 over gloo.  Each rank runs the oracle on its shard of the env ids (the product's
sharding rule, paper_2606_11440_b200/sharding.py), the four sums of SURVEY 8(e) are all-reduced (the product's one
collective, sharding.allreduce_sums), and the result must equal the unsharded run: trajectories column for column
(R2: draws keyed by global env id), C-bar / U-bar / sigma_U to rounding.  What each rank does with the job-wide sums on
the GPU (im_returns_finish) is covered by tests/test_gpu_parity.py::test_two_shards_normalise_like_one_context."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from helpers import tiny_spec
from im_workload import make_policy_blob
from paper_2606_11440_b200.sharding import allreduce_sums, shard_range, shard_spec


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spec():
    return tiny_spec(n_envs=11, N=2, n_ticks=160, qcap=16, rcap=48, rate_tick=[0.2, 0.45, 0.3], slots=3, budget=(30, 150), seed=5)


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle as O
    full = _spec()
    blob = make_policy_blob(full, seed=2)
    mine = shard_spec(full, rank, world)
    base, cnt = shard_range(full.n_envs, rank, world)
    o = O.Oracle(mine, seed=7, env_ids=np.arange(base, base + cnt, dtype=np.uint32))
    o.rollout(blob, full.n_ticks, n_threads=1)
    o.returns(0.97, 0.9, 0.4)
    # the rank's four sums, from its own query log and cost array (what IM_TEL_SUMS holds on the GPU)
    q = o.queries()
    U = ((q["info"] >> 16) & 1).astype(np.float64) - 0.4 * q["sojourn"].astype(np.float64) / (q["info"] & 0xFFFF)
    mine = np.array([o.cost().astype(np.float64).sum(), U.size, U.sum(), (U * U).sum()])
    tot = allreduce_sums(mine, device="cpu")
    ubar = tot[2] / tot[1]
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), rew=o.rew(), cost=o.cost(), adv=o.adv(), base=base, cnt=cnt,
             cbar=tot[0] / tot[1], ubar=ubar, usigma=np.sqrt(max(tot[3] / tot[1] - ubar * ubar, 0.0)), n_final=int(tot[1]))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_range_covers_everything_once():
    for n, w in ((11, 2), (262144, 8), (7, 7), (100, 3)):
        got = [shard_range(n, r, w) for r in range(w)]
        assert got[0][0] == 0 and sum(c for _, c in got) == n
        for (b0, c0), (b1, _) in zip(got, got[1:]):
            assert b0 + c0 == b1
        assert max(c for _, c in got) - min(c for _, c in got) <= 1


def test_shard_spec_sizes_caps_from_the_shards_own_levels():
    """A utilisation sweep over contiguous shards: the last shard carries more load than the first, and its log
    capacities follow; a capacity of 0 (library default) stays 0."""
    full = tiny_spec(n_envs=64, N=2, n_ticks=100, qcap=16, rcap=64, rate_tick=[0.1, 0.2, 0.4, 0.8], slots=3, seed=5)
    full = full.with_(env_level=(np.arange(64) * 4 // 64).astype(np.uint8), log_cap_exec=100000, log_cap_plan=0)
    first, last = shard_spec(full, 0, 4), shard_spec(full, 3, 4)
    assert last.log_cap_exec > 3 * first.log_cap_exec and first.log_cap_plan == 0 == last.log_cap_plan
    assert first.env_id_base == 0 and last.env_id_base == 48 and first.n_envs == last.n_envs == 16


def test_two_ranks_over_gloo_equal_the_unsharded_run(tmp_path):
    from oracle import oracle as O
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    full = _spec()
    blob = make_policy_blob(full, seed=2)
    o = O.Oracle(full, seed=7)
    o.rollout(blob, full.n_ticks, n_threads=1)
    o.returns(0.97, 0.9, 0.4)
    ref = o.scalars()
    rew, cost, adv = o.rew(), o.cost(), o.adv()
    for r in range(world):
        d = np.load(os.path.join(str(tmp_path), f"rank{r}.npz"))
        b, c = int(d["base"]), int(d["cnt"])
        assert np.array_equal(d["rew"], rew[:, b:b + c]) and np.array_equal(d["cost"], cost[:, b:b + c])
        assert np.array_equal(d["adv"], adv[:, b:b + c])
        assert int(d["n_final"]) == ref["n_final"] and ref["n_final"] > 50
        for k in ("cbar", "ubar", "usigma"):
            assert abs(float(d[k]) - ref[k]) <= 1e-12 * max(1.0, abs(ref[k])), (k, float(d[k]), ref[k])
