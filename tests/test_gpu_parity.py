"""GPU parity tests proper: the CUDA path through the C ABI vs the oracle, element by element."""
import numpy as np
import pytest

from helpers import tiny_spec
from im_workload import make_policy_blob, make_pool_spec
from parity import compare_chunk, compare_returns, finish_stats

pytestmark = pytest.mark.gpu

FLAGS_F32 = 1          # LOG_DECISIONS
FLAGS_BF16 = 3         # + LOG_LOGITS


def _run(spec, seed, chunks, blob=None, env_ids=None, gamma=0.99, lam=0.95, mu=0.5, weight_scale=1.0):
    from oracle import oracle as O
    from paper_2606_11440_b200 import InfraMind
    bf16 = spec.policy_dtype == 1
    blob = make_policy_blob(spec, seed=0, scale=weight_scale) if blob is None else blob
    if env_ids is None:
        env_ids = np.arange(spec.n_envs, dtype=np.uint32) + np.uint32(spec.env_id_base)
    gpu = InfraMind(spec, seed=seed, debug_flags=FLAGS_BF16 if bf16 else FLAGS_F32)
    orc = O.Oracle(spec, seed=seed, env_ids=env_ids, keep_logits=False)
    stats = {}
    for n in chunks:
        compare_chunk(gpu, orc, env_ids, n, blob, bf16, stats)
    finish_stats(orc, stats, bf16)
    compare_returns(gpu, orc, env_ids, gamma, lam, mu, bf16, whole_batch=(len(env_ids) == spec.n_envs))
    csum = gpu.counters().sum(axis=0)
    stats.update(arrivals=int(csum[0]), dropped=int(csum[1]), finished=int(csum[2]), preemptions=int(csum[7]), missed=int(csum[4]))
    gpu.close()
    return stats


def test_cfg1_full_every_tick():
    """configs[0]: E=64, 5 models, 200 ticks, fp32 policy; state compared after every tick."""
    spec = make_pool_spec(1)
    st = _run(spec, seed=0, chunks=[1] * 200)
    assert st["decisions"] > 2000


def test_cfg1_scaled_weights_chunked():
    spec = make_pool_spec(1)
    st = _run(spec, seed=3, chunks=[7, 50, 1, 100, 42], weight_scale=4.0)
    assert st["decisions"] > 2000


def test_cfg2_slice():
    """configs[1] slice: 256 of the 4096 envs (E-invariance: env e depends only on its global id), 600 ticks."""
    spec = make_pool_spec(2, n_envs=256, n_ticks=600)
    _run(spec, seed=0, chunks=[100] * 6)


def test_cfg3_overload_bf16_slice():
    """configs[2] slice: 8 models, preemption, overload rho=1.2, bf16 64->128 policy, teacher-forced sampling."""
    spec = make_pool_spec(3, n_envs=160, n_ticks=500)
    _run(spec, seed=0, chunks=[1] * 20 + [80] * 6)


def test_cfg4_heterogeneous_bf16_slice():
    """configs[3] slice: 16 models, prefill, input tokens, swept utilisation, bf16 128->256 policy."""
    spec = make_pool_spec(4, n_envs=192, n_ticks=400)
    _run(spec, seed=0, chunks=[1] * 10 + [65] * 6)


def test_cfg5_bimodal_bf16_slice():
    spec = make_pool_spec(5, n_envs=130, n_ticks=300)   # ragged: 130 is not a multiple of any tile size
    _run(spec, seed=1, chunks=[100] * 3)


def test_fcfs_and_episodes_and_miss_cost():
    """FCFS scheduling, episode resets (done flags cut GAE), cost_mode=1."""
    spec = tiny_spec(n_envs=37, N=3, n_ticks=240, qcap=32, rcap=128, rate_tick=0.35, slots=2, sched_mode=0,
                     episode_ticks=60, cost_mode=1, f_in=32, hidden=64, budget=(20, 120))
    _run(spec, seed=5, chunks=[60, 1, 59, 120])


def test_t9_bimodal_budgets_edf_vs_fcfs_single_server():
    """PAPER.md:179 (Table 3, "w/o EDF"), qualitative: one stable single-slot server, budgets 100 / 1000 ticks.
    Both orders are bit-exact against the oracle, and the CUDA path's own counters show fewer misses under EDF."""
    from helpers import forced_single_blob
    kw = dict(n_envs=35, N=1, n_ticks=1500, qcap=64, rcap=256, rate_tick=0.025, slots=1, budget=(100, 100), seed=3,
              rates=[40], f_in=32, hidden=64)
    missed = []
    for mode in (0, 1):
        spec = tiny_spec(sched_mode=mode, **kw).with_(
            mix_thresh=0x80000000, mix_lo=np.array([100, 1000], dtype=np.uint32),
            mix_hi=np.array([100, 1000], dtype=np.uint32), budget_norm_ticks=1000)
        st = _run(spec, seed=5, chunks=[700, 800], blob=forced_single_blob(spec))
        assert st["dropped"] == 0
        missed.append(st["missed"])
    assert missed[1] < 0.75 * missed[0]


def test_tiny_queue_preemption_fp32():
    """Small KV with preemption on an fp32 policy: exercises H (evictions) with bit-exact decisions."""
    spec = tiny_spec(n_envs=33, N=2, n_ticks=300, qcap=32, rcap=128, rate_tick=0.4, slots=8, kv_preempt=1, kv_cap=700,
                     budget=(50, 400), medians=(100, 200, 300), f_in=32, hidden=64, seed=3)
    st = _run(spec, seed=6, chunks=[1] * 50 + [250])
    assert st["decisions"] > 1000


def test_env_id_base_shard_equals_full():
    """Multi-GPU sharding rule: a shard with env_id_base reproduces the same envs of the full run."""
    from paper_2606_11440_b200 import InfraMind
    full = make_pool_spec(1)
    blob = make_policy_blob(full)
    a = InfraMind(full, seed=0, debug_flags=1)
    a.rollout(blob, 120)
    shard = full.with_(n_envs=24, env_id_base=40, env_level=full.env_level[40:64].copy())
    b = InfraMind(shard, seed=0, debug_flags=1)
    b.rollout(blob, 120)
    assert np.array_equal(a.state()[40:64], b.state())
    assert np.array_equal(a.rew()[:, 40:64], b.rew()) and np.array_equal(a.val()[:, 40:64], b.val())
    a.close(); b.close()


def test_two_shards_normalise_like_one_context():
    """SURVEY 8(e) / PAPER.md:127-129: an env-sharded job must produce the single-GPU result.  Two contexts with
    env_id_base 0 and E/2 stand in for two ranks: their IM_TEL_SUMS are added (the job's one all-reduce) and handed
    to im_returns_finish; every rank's UNORM and scalars then equal those of one context over all envs."""
    from paper_2606_11440_b200 import InfraMind
    full = make_pool_spec(1, n_envs=64, n_ticks=200)
    blob = make_policy_blob(full)
    mu = 0.5
    one = InfraMind(full, seed=0, debug_flags=1)
    one.rollout(blob, 200); one.returns(0.99, 0.95, mu)
    ref_q, ref_s = one.queries(unorm=True), one.scalars()
    ref_sums = one.sums()
    assert abs(ref_sums[0] - ref_s["sum_cost"]) < 1e-9 and int(ref_sums[1]) == ref_s["n_final"] > 200
    parts = []
    for base in (0, 32):
        sh = full.with_(n_envs=32, env_id_base=base, env_level=full.env_level[base:base + 32].copy())
        g = InfraMind(sh, seed=0, debug_flags=1)
        g.rollout(blob, 200); g.returns(0.99, 0.95, mu)
        parts.append(g)
    local = [g.queries(unorm=True)["unorm"].copy() for g in parts]
    total = parts[0].sums() + parts[1].sums()
    assert np.allclose(total, ref_sums, rtol=1e-12, atol=1e-9)
    # records with the same (env, arrive, sojourn, info) have the same utility: sort on those and compare in that order
    order = lambda q: np.lexsort((q["info"], q["sojourn"], q["arrive"], q["env"]))
    ro = order(ref_q)
    moved = 0.0
    for g, loc in zip(parts, local):
        g.returns_finish(total)
        q, sc = g.queries(unorm=True), g.scalars()
        for k in ("cbar", "ubar", "usigma"):
            assert abs(sc[k] - ref_s[k]) <= 1e-9 * max(1.0, abs(ref_s[k])), k
        assert sc["n_final"] == ref_s["n_final"]
        mine = ref_q["env"][ro] // 32 == (0 if g is parts[0] else 1)        # this shard's envs in the full run
        go = order(q)
        assert np.array_equal(q["sojourn"][go], ref_q["sojourn"][ro][mine]) and np.array_equal(q["info"][go], ref_q["info"][ro][mine])
        assert np.max(np.abs(q["unorm"][go] - ref_q["unorm"][ro][mine])) <= 1e-6
        moved = max(moved, float(np.max(np.abs(q["unorm"] - loc))))
        g.close()
    assert moved > 1e-4                      # the shard-local normalisation really was different
    one.close()


def test_determinism_and_split():
    from paper_2606_11440_b200 import InfraMind
    spec = make_pool_spec(3, n_envs=96, n_ticks=200)
    blob = make_policy_blob(spec)
    g = InfraMind(spec, seed=2, debug_flags=1)
    g.rollout(blob, 200)
    s1, c1, r1 = g.state(), g.counters(), g.rew()
    g.reset(); g.rollout(blob, 200)
    assert np.array_equal(s1, g.state()) and np.array_equal(c1, g.counters()) and np.array_equal(r1, g.rew())
    g.reset(); g.rollout(blob, 77); ra = g.rew(); g.rollout(blob, 123); rb = g.rew()
    assert np.array_equal(s1, g.state()) and np.array_equal(np.concatenate([ra, rb]), r1)
    g.close()


def test_queue_order_matches_oracle():
    """IM_TEL_QUEUE_ORDER (segmented bitonic sort kernel) vs the oracle's repeated arg-min (R20)."""
    from oracle import oracle as O
    from paper_2606_11440_b200 import InfraMind
    for mode in (0, 1):
        spec = make_pool_spec(3, n_envs=48, n_ticks=150).with_(sched_mode=mode)
        blob = make_policy_blob(spec)
        g = InfraMind(spec, seed=1, debug_flags=0)
        o = O.Oracle(spec, seed=1)
        g.rollout(blob, 150); o.rollout(blob, 150)
        qo = g.queue_order()
        N, tot = spec.n_models, 0
        for e in range(48):
            off = qo[e, : N + 1]
            for k in range(N):
                ref = o.queue_order(e, k, 150)
                got = qo[e, N + 1 + off[k]: N + 1 + off[k + 1]]
                assert np.array_equal(got, ref)
                tot += len(ref)
        assert tot > 1000
        g.close()


def test_error_paths():
    from paper_2606_11440_b200 import InfraMind, IMError
    spec = make_pool_spec(1, n_envs=8, n_ticks=10)
    g = InfraMind(spec, seed=0, debug_flags=1)
    with pytest.raises(IMError) as ei:
        g.returns(0.99, 0.95, 0.5)
    assert ei.value.code == -5
    with pytest.raises(IMError) as ei:
        g.rollout(make_policy_blob(spec), 11)
    assert ei.value.code == -6
    bad = make_policy_blob(make_pool_spec(3, n_envs=8, n_ticks=10))
    with pytest.raises(IMError) as ei:
        g.rollout(bad, 5)
    assert ei.value.code == -2
    g.rollout(make_policy_blob(spec), 5)
    with pytest.raises(IMError) as ei:
        g.adv()
    assert ei.value.code == -5
    g.close()
