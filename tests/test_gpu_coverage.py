"""GPU parity at the coverage SURVEY §8(c) step 5 asks for (through the C ABI, vs the oracle, element by element).

* configs[2..4] on >= 2048 env ids SPREAD OVER ALL ARRIVAL LEVELS: the utilisation sweep assigns level floor(64 e / E), so
  a slice of the first few hundred ids only ever sees the lightest level.  Every draw is keyed by the global env id (R2),
  so a small context with env_id_base = b reproduces envs b .. b + w of the full run: many such contexts, one per level
  block, cover the sweep (overload included) at a size the oracle replays in seconds.
* configs[1] in full: E = 4096 envs x T = 2000 ticks.
* configs[2] and configs[3] through all eight im_rollout(500) calls to tick 4000 (16-bit clock fields, 13-bit relative
  ticks of the row lists, ring wrap of the logs) on sampled ranges inside a FULL-E context, as test_gpu_fullsize.py
  does for configs[4].
* IM_TEL_TABLES byte for byte; the row-list ring without a decision log (debug_flags = 0) under arrival bursts.
"""
import numpy as np
import pytest

from helpers import tiny_spec
from im_workload import CONFIGS, make_policy_blob, make_pool_spec
from parity import compare_chunk, compare_returns, finish_stats

pytestmark = pytest.mark.gpu


def _small(full, base, width, T):
    cap = width * T * 48 + 4096
    return full.with_(n_envs=width, env_id_base=base, env_level=full.env_level[base:base + width].copy(), n_ticks=T,
                      log_cap_exec=cap, log_cap_plan=cap, log_cap_query=cap)


def _spread(cfg, n_ctx, width, chunks, seed=0):
    """n_ctx small contexts of `width` envs whose bases are spread evenly over the config's full env range."""
    from oracle import oracle as O
    from paper_2606_11440_b200 import InfraMind
    full = make_pool_spec(cfg)
    E, T = full.n_envs, sum(chunks)
    blob = make_policy_blob(full, seed=0)
    levels, tot = set(), dict(decisions=0, dropped=0, preempt=0, finished=0)
    for i in range(n_ctx):
        base = min(i * E // n_ctx + (E // n_ctx) // 2, E - width)          # the middle of the i-th stretch
        sp = _small(full, base, width, T)
        env_ids = np.arange(base, base + width, dtype=np.uint32)
        g = InfraMind(sp, seed=seed, debug_flags=3)
        o = O.Oracle(sp, seed=seed, env_ids=env_ids, keep_logits=False)
        st = {}
        for n in chunks:
            compare_chunk(g, o, env_ids, n, blob, True, st)
        finish_stats(o, st, True)
        compare_returns(g, o, env_ids, 0.99, 0.95, 0.5, True, whole_batch=True)
        c = g.counters().sum(axis=0)
        tot["decisions"] += st["decisions"]; tot["dropped"] += int(c[1]); tot["preempt"] += int(c[7]); tot["finished"] += int(c[2])
        levels.update(np.unique(sp.env_level).tolist())
        g.close(); o.close()
    return levels, tot


def test_cfg3_2048_ids_spread_over_the_range():
    """configs[2]: one level (rho = 1.2), 2048 env ids taken from 16 stretches of the 65536."""
    levels, tot = _spread(3, n_ctx=16, width=128, chunks=[150, 150])
    assert levels == {0} and tot["decisions"] > 200000 and tot["preempt"] > 0


def test_cfg4_2048_ids_over_all_64_levels():
    """configs[3]: utilisation swept 0.2 .. 1.3 across env blocks - one context per level, the overloaded half included."""
    levels, tot = _spread(4, n_ctx=64, width=32, chunks=[200, 200])
    assert levels == set(range(64)) and tot["decisions"] > 200000 and tot["preempt"] > 0


def test_cfg5_2048_ids_over_all_64_levels():
    """configs[4]: the same sweep with bimodal budgets."""
    levels, tot = _spread(5, n_ctx=64, width=32, chunks=[150, 150], seed=2)
    assert levels == set(range(64)) and tot["decisions"] > 150000 and tot["finished"] > 20000


def test_cfg2_full_size():
    """configs[1] as BASELINE.json states it: all 4096 envs, 2000 ticks, every decision recomputed by the oracle (fp32)."""
    from oracle import oracle as O
    from paper_2606_11440_b200 import InfraMind
    spec = make_pool_spec(2)
    assert (spec.n_envs, spec.n_ticks) == (4096, 2000)
    blob = make_policy_blob(spec, seed=0)
    env_ids = np.arange(4096, dtype=np.uint32)
    g = InfraMind(spec, seed=0, debug_flags=1)
    o = O.Oracle(spec, seed=0, env_ids=env_ids, keep_logits=False)
    st = {}
    for n in (500, 500, 500, 500):
        compare_chunk(g, o, env_ids, n, blob, False, st, check_state=True)
    finish_stats(o, st, False)
    compare_returns(g, o, env_ids, 0.99, 0.95, 0.5, False, whole_batch=True)
    assert st["decisions"] > 3_000_000
    g.close(); o.close()


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_context_through_eight_chunks_to_tick_4000(cfg):
    """configs[2] / configs[3] in bench.py's launch configuration: E = 65536 / 131072, eight im_rollout(500) calls with
    persistent state.  Sampled env ranges (spread over the levels) are re-run as small contexts against the oracle
    for all 4000 ticks; after every call their trajectory rows and counters must equal the same columns of the
    full-size run bit for bit."""
    import torch
    from oracle import oracle as O
    from paper_2606_11440_b200 import InfraMind, IM_TEL_REW, IM_TEL_COST, IM_TEL_VAL, IM_TEL_MISS
    full = make_pool_spec(cfg)
    E, T, chunk = full.n_envs, full.n_ticks, full.max_ticks
    assert T == 4000 and chunk == 500 and E == CONFIGS[cfg]["E"]
    blob = make_policy_blob(full, seed=0)
    width = 20
    bases = [0, E // 3 + 11, (2 * E) // 3 + 5, E - width] if cfg == 3 else [3, E // 2 - 7, (3 * E) // 4 + 1, E - width]
    cols = torch.cat([torch.arange(b, b + width) for b in bases]).to("cuda")
    gpu = InfraMind(full, seed=0, debug_flags=1)          # bench.py's configuration
    snaps, ctrs = [], None
    for k in range(T // chunk):
        gpu.rollout(blob, chunk)
        gpu.sync()
        snaps.append({name: gpu.device_tensor(what, dt).view(-1, E)[:chunk, cols].cpu().numpy()
                      for name, what, dt in (("rew", IM_TEL_REW, torch.float32), ("cost", IM_TEL_COST, torch.float32),
                                             ("val", IM_TEL_VAL, torch.float32), ("miss", IM_TEL_MISS, torch.uint8))})
    ctrs = gpu.counters().astype(np.int64)
    assert gpu.scalars()["tick"] == 4000
    gpu.close()
    del gpu
    torch.cuda.empty_cache()
    for i, b in enumerate(bases):
        sl = slice(i * width, (i + 1) * width)
        sp = _small(full, b, width, chunk).with_(max_ticks=chunk)
        env_ids = np.arange(b, b + width, dtype=np.uint32)
        g = InfraMind(sp, seed=0, debug_flags=3)
        o = O.Oracle(sp, seed=0, env_ids=env_ids, keep_logits=False)
        st = {}
        for k in range(T // chunk):
            compare_chunk(g, o, env_ids, chunk, blob, True, st, check_state=(k % 4 == 3))
            assert np.array_equal(g.rew(), snaps[k]["rew"][:, sl]) and np.array_equal(g.cost(), snaps[k]["cost"][:, sl])
            assert np.array_equal(g.miss(), snaps[k]["miss"][:, sl]) and np.array_equal(g.val()[:chunk], snaps[k]["val"][:, sl])
        finish_stats(o, st, True)
        assert np.array_equal(g.counters().astype(np.int64), ctrs[b:b + width])
        g.close(); o.close()


def test_tables_read_back_byte_for_byte():
    """SURVEY 8(c) parity protocol step 1: IM_TEL_TABLES == the harness tables (no libm difference can enter the dynamics)."""
    from paper_2606_11440_b200 import InfraMind, IM_TEL_TABLES
    for cfg in (1, 5):
        spec = make_pool_spec(cfg, n_envs=64, n_ticks=4)
        g = InfraMind(spec, seed=0, debug_flags=0)
        raw = g.read(IM_TEL_TABLES, np.uint32)
        assert raw.size == 2048 + spec.n_levels * 32
        assert np.array_equal(raw[:1024], spec.out_tok_mult_q16.astype(np.uint32))
        assert np.array_equal(raw[1024:2048], np.zeros(1024, np.uint32) if spec.in_tok_table is None else spec.in_tok_table.astype(np.uint32))
        assert np.array_equal(raw[2048:], spec.arr_cdf.astype(np.uint32).ravel())
        g.close()


def test_row_rings_without_a_decision_log_hold_a_bursty_tick():
    """debug_flags = 0 (the ABI's default): the work lists are rings that hold one tick's rows and log_cap_exec / plan are
    ignored.  Poisson(14) arrivals per tick give bursts of 20+ queries (60+ executor rows) per env in one tick; the run
    must either stay bit-exact against the oracle (fp32 policy: the oracle recomputes every decision itself) or report
    IM_ERR_CAPACITY - never lose or duplicate a decision silently."""
    from oracle import oracle as O
    from paper_2606_11440_b200 import InfraMind, IMError
    spec = tiny_spec(n_envs=70, N=2, n_ticks=60, qcap=256, rcap=1024, rate_tick=14.0, slots=64, rates=[200, 200], budget=(5, 30),
                     medians=(4, 8, 12), f_in=32, hidden=32, seed=4).with_(log_cap_exec=64, log_cap_plan=64)
    blob = make_policy_blob(spec)
    g = InfraMind(spec, seed=9, debug_flags=0)
    o = O.Oracle(spec, seed=9)
    try:
        for n in (1, 9, 50):
            g.rollout(blob, n)
            o.rollout(blob, n, n_threads=8)
            oc = o.counters(); oc[:, 14] = 0
            assert np.array_equal(g.counters(), oc) and np.array_equal(g.state(), o.state())
            assert np.array_equal(g.rew(), o.rew()) and np.array_equal(g.val(), o.val())
        assert g.counters()[:, 0].sum() > 70 * 60 * 12
    except IMError as err:
        assert err.code == -6
    g.close(); o.close()
