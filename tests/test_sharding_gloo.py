"""N > 1 path on CPU: world_size 2 over gloo.  Each rank runs the oracle on its shard of the env ids (the product's
sharding rule, paper_2606_11440_b200/sharding.py), the four sums are all-reduced, and the result must equal the
unsharded run: trajectories column for column (R2: draws keyed by global env id), C-bar / U-bar / sigma_U to rounding."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from helpers import tiny_spec
from im_workload import make_policy_blob
from paper_2606_11440_b200.sharding import allreduce_scalars, combine_sums, partial_sums, shard_range, shard_spec


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
    red = allreduce_scalars(o.scalars(), device="cpu")
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), rew=o.rew(), cost=o.cost(), adv=o.adv(), base=base, cnt=cnt,
             cbar=red["cbar"], ubar=red["ubar"], usigma=red["usigma"], n_final=red["n_final"])
    dist.barrier()
    dist.destroy_process_group()


def test_shard_range_covers_everything_once():
    for n, w in ((11, 2), (262144, 8), (7, 7), (100, 3)):
        got = [shard_range(n, r, w) for r in range(w)]
        assert got[0][0] == 0 and sum(c for _, c in got) == n
        for (b0, c0), (b1, _) in zip(got, got[1:]):
            assert b0 + c0 == b1
        assert max(c for _, c in got) - min(c for _, c in got) <= 1


def test_combine_sums_matches_direct_moments():
    rng = np.random.default_rng(0)
    u = rng.normal(0.3, 0.5, size=1000)
    parts = [dict(sum_cost=float(i + 1), n_final=len(x), ubar=float(x.mean()), usigma=float(x.std())) for i, x in enumerate(np.split(u, [300, 650]))]
    tot = np.sum([partial_sums(p) for p in parts], axis=0)
    c = combine_sums(*tot)
    assert c["n_final"] == 1000 and abs(c["ubar"] - u.mean()) < 1e-12 and abs(c["usigma"] - u.std()) < 1e-12 and abs(c["cbar"] - 6.0 / 1000) < 1e-15


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
