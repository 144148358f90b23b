"""GPU parity on the degenerate and extreme cases of the path (through the C ABI, vs the oracle, element by element)."""
import numpy as np
import pytest

from helpers import tiny_spec
from im_workload import make_policy_blob
from test_gpu_parity import _run

pytestmark = pytest.mark.gpu


def test_no_arrivals_everything_stays_zero():
    """Empty input: arrival rate 0 => no query, no decision, all-zero trajectories; V[t] is the critic on a zero snapshot."""
    from paper_2606_11440_b200 import InfraMind
    spec = tiny_spec(n_envs=19, N=3, n_ticks=40, qcap=32, rcap=128, rate_tick=0.0, slots=4, f_in=32, hidden=32)
    _run(spec, seed=1, chunks=[1, 39])
    g = InfraMind(spec, seed=1, debug_flags=1)
    g.rollout(make_policy_blob(spec), 40)
    assert not g.rew().any() and not g.cost().any() and not g.miss().any() and not g.counters().any()
    assert np.all(g.val() == g.val()[0, 0])
    g.close()


def test_full_query_table_drops_and_long_waiting_list():
    """Overload far beyond capacity: the query table fills (tail drops, R9: miss + cost 1.0 per drop), the waiting list
    reaches its bound of 3 calls per live query, admission scans a long list every tick."""
    spec = tiny_spec(n_envs=21, N=2, n_ticks=160, qcap=32, rcap=128, rate_tick=3.0, slots=2, rates=[60, 45], budget=(20, 90),
                     medians=(200, 400, 800), f_in=32, hidden=32, seed=8)
    st = _run(spec, seed=2, chunks=[1] * 30 + [130])
    assert st["decisions"] > 500 and st["dropped"] > 1000 and st["finished"] > 5


def test_sixteen_models_extreme_slot_counts_and_largest_tables():
    """N = 16 with slot counts 1 .. 64 (a lane's 8 slots never straddle two models), qcap = 1024 (12-bit request ids),
    KV pressure with preemption on a few models, prefill, fp32 policy (decisions bit-exact)."""
    slots = [1, 64, 8, 3, 17, 64, 2, 40, 9, 1, 33, 5, 64, 12, 7, 24]
    kv = [4000, 30000, 6000, 5000, 9000, 25000, 4000, 20000, 6000, 4000, 15000, 5000, 28000, 8000, 5000, 12000]
    spec = tiny_spec(n_envs=9, N=16, n_ticks=150, qcap=1024, rcap=3072, rate_tick=2.2, slots=slots, kv_cap=kv, kv_preempt=1,
                     budget=(30, 400), medians=(150, 500, 1200), in_tok=600, prefill=900, f_in=64, hidden=32, seed=12)
    st = _run(spec, seed=3, chunks=[1] * 10 + [140])
    assert st["decisions"] > 500 and st["preemptions"] > 0


def test_single_model_single_slot():
    """N = 1, S = 1: the M/M/1 shape of pin P6 on the GPU path (every admission waits for the one slot)."""
    spec = tiny_spec(n_envs=17, N=1, n_ticks=300, qcap=64, rcap=256, rate_tick=0.06, slots=1, rates=[80], budget=(100, 900),
                     medians=(40, 80, 160), f_in=32, hidden=16, seed=4)
    _run(spec, seed=4, chunks=[300])


def test_clock_limit_is_an_error_not_a_wraparound():
    """Device state keeps absolute ticks in 16 bits: im_rollout refuses to run past tick + budget >= 65536."""
    from paper_2606_11440_b200 import InfraMind, IMError
    spec = tiny_spec(n_envs=4, N=1, n_ticks=8000, qcap=32, rcap=128, rate_tick=0.01, slots=2, f_in=32, hidden=16, budget=(10, 1000))
    g = InfraMind(spec, seed=0, debug_flags=0)
    blob = make_policy_blob(spec)
    for _ in range(8):
        g.rollout(blob, 8000)
    with pytest.raises(IMError) as ei:
        g.rollout(blob, 8000)           # 64000 + 8000 + 1000 >= 65536
    assert ei.value.code == -6
    g.reset()
    g.rollout(blob, 100)                # the clock restarts with im_reset
    g.close()


def test_arrival_bursts_of_sixteen_and_more():
    """Poisson(14) arrivals per tick with short calls and a large table: bursts of 16..31 queries in one tick are common,
    i.e. more arrivals than a group has lanes (the second iteration of the arrival loop and its separately drawn
    budgets, R7/R8)."""
    from paper_2606_11440_b200 import InfraMind
    spec = tiny_spec(n_envs=11, N=2, n_ticks=50, qcap=256, rcap=1024, rate_tick=14.0, slots=64, rates=[200, 200], budget=(5, 30),
                     medians=(4, 8, 12), f_in=32, hidden=32, seed=4)
    cap = (64 + spec.n_envs) * spec.n_ticks * 80
    spec = spec.with_(log_cap_exec=cap, log_cap_plan=cap, log_cap_query=cap)
    st = _run(spec, seed=9, chunks=[1] * 10 + [40])
    assert st["arrivals"] > 11 * 50 * 12
    # some tick of some env took sixteen or more queries at once: the planner log holds one row per accepted arrival
    g = InfraMind(spec, seed=9, debug_flags=1)
    before = g.counters()[:, 10].astype(np.int64)
    burst = 0
    for _ in range(50):
        g.rollout(make_policy_blob(spec), 1)
        now = g.counters()[:, 10].astype(np.int64)
        burst = max(burst, int((now - before).max()))
        before = now
    g.close()
    assert burst >= 16


def test_device_blob_of_another_spec_is_rejected():
    """A DEVICE blob cannot be checked on the host without a synchronisation: its header is checked on the device and the
    mismatch surfaces as IM_ERR_BAD_SPEC at the next read; ADV / RET device pointers need im_returns first."""
    import torch
    from im_workload import make_pool_spec
    from paper_2606_11440_b200 import InfraMind, IMError, IM_TEL_ADV
    spec = make_pool_spec(1, n_envs=8, n_ticks=10)
    g = InfraMind(spec, seed=0, debug_flags=1)
    with pytest.raises(IMError) as ei:
        g.device_tensor(IM_TEL_ADV, torch.float32)
    assert ei.value.code == -5
    other = make_policy_blob(make_pool_spec(3, n_envs=8, n_ticks=10))
    good = make_policy_blob(spec)
    bad = torch.from_numpy(np.resize(other, good.size)).cuda()
    g.rollout(bad, 2)
    with pytest.raises(IMError) as ei:
        g.rew()
    assert ei.value.code == -2
    g.close()
    # a pinned host blob may be overwritten right after the call returns
    g = InfraMind(spec, seed=0, debug_flags=1)
    pin = torch.from_numpy(good.copy()).pin_memory()
    g.rollout(pin.numpy(), 10)
    pin.zero_()
    a = g.rew().copy(); c1 = g.counters().copy()
    g.reset(); g.rollout(good, 10)
    assert np.array_equal(a, g.rew()) and np.array_equal(c1, g.counters())
    g.close()


@pytest.mark.parametrize("sched_mode,kv_preempt", [(1, 0), (0, 0), (1, 1)])
def test_direct_admission_borderline_cases(sched_mode, kv_preempt):
    """k_sim admits a call straight from its issue record when it is its model's only issue of the tick and the queue is
    empty.  Debate with K = 4 issues three calls in ONE tick, forced onto two models with two slots each and a KV capacity
    that fits one or two requests: same-model issues in one tick (must go through the list, smallest key first, stop at
    the first misfit), lone issues that do not fit (must wait), lone issues that fit (admitted directly), all interleaved
    with completions and, with kv_preempt, evictions back into the list.  Compared with the oracle after EVERY tick
    (state dump included), EDF and FCFS."""
    from helpers import planner_bias_blob
    N = 2
    spec = tiny_spec(n_envs=37, N=N, n_ticks=220, qcap=32, rcap=128, rate_tick=[0.05, 0.25, 0.6], slots=2, rates=[90, 140],
                     kv_cap=[700, 1100], kv_preempt=kv_preempt, sched_mode=sched_mode, budget=(20, 120), medians=(60, 120, 240),
                     in_tok=300, prefill=400, f_in=32, hidden=16, seed=21)
    bias = np.full(3 * N, -40.0)
    bias[[0, 1, 3, 4, 5]] = 0.0                               # both models, several depths: uniform among them
    st = _run(spec, seed=6, chunks=[1] * 220, blob=planner_bias_blob(spec, topo=2, count=4, exec_bias=bias))
    assert st["decisions"] > 3000 and st["finished"] > 50
    if kv_preempt:
        assert st["preemptions"] > 0


def test_random_access_probe_orders_the_access_shapes():
    """libimprobe (bench.py's ceilings for k_sim): a full-sector 256-bit store must beat a half-sector store clearly (the
    reason the running-slot records are 32 bytes), and every rate is a positive, sane number."""
    from paper_2606_11440_b200.probe import random_access_rates
    r = random_access_rates(gib=4, rounds=16)
    assert set(r) == {"read16", "write16", "write32", "rmw4"}
    assert all(1.0 < v < 2000.0 for v in r.values()), r
    assert r["write32"] > 1.3 * r["write16"] and r["read16"] > r["write16"] > r["rmw4"], r
