"""Pins of the oracle parts the round-1 review found unpinned (VERDICT.md "Parity unpinned" 1-6).  All `-m "not gpu"`.

Each test compares the oracle with something it did not compute: an exact integer recomputation from its logs, a
closed-form probability, a stage table typed here from DESIGN.md R17, a brute-force replay of one admission from the
previous tick's state dump.  Each docstring names the oracle mutation the test was seen to fail under.
"""
import math

import numpy as np

from helpers import decode_state, forced_single_blob, planner_bias_blob, tiny_spec, ST_RUN, ST_WAIT
from im_workload import make_policy_blob

CN = {n: i for i, n in enumerate(
    ["arrivals", "dropped", "finished", "solved", "missed", "calls_issued", "calls_done", "preemptions", "sum_sojourn",
     "sum_live_mid", "plans", "exec_decisions", "sum_running", "sum_waiting", "near_boundary", "abandoned"])}


# --------------------------------------------------------------------------------- (a) cost value
def test_cost_is_call_latency_over_the_querys_budget(orc):
    """C_k = l_k / beta.  Chains of 3 calls on an uncontended pool: call j is issued at the tick of its
    decision and completes the tick before the next call of its query is issued (the last one at the finalisation
    tick), so every l_k follows from the decision log and the query log alone.  cost[t, e] must equal the sum over
    the calls completing in t of floor(l_k * 2^16 / beta) * 2^-16 with beta the QUERY's budget (R28), exactly.
    Fails under: dividing by budget_norm_ticks instead of the query's budget; l = t - issue (off by one); cost
    attributed to the issue tick."""
    T = 500
    spec = tiny_spec(n_envs=12, N=2, n_ticks=T, qcap=64, rcap=192, rate_tick=0.05, slots=64, rates=[90, 140],
                     budget=(40, 400), medians=(30, 70, 150))
    o = orc.Oracle(spec, seed=4)
    o.rollout(planner_bias_blob(spec, topo=1, count=3), T)
    q, d = o.queries(), o.decisions(1)
    assert o.counters()[:, CN["dropped"]].sum() == 0 and q["sojourn"].size > 100
    expect = np.zeros((T, 12), dtype=np.int64)           # Q16
    dirty = np.zeros((T, 12), dtype=bool)                # ticks that may hold calls of a query this test cannot attribute
    starts = {}
    for j in range(d["t"].size):
        if d["agent"][j] == 0:
            starts.setdefault((int(d["env_local"][j]), int(d["t"][j])), []).append(int(d["q"][j]))
    calls = {}
    for j in range(d["t"].size):
        calls.setdefault((int(d["env_local"][j]), int(d["q"][j])), []).append((int(d["t"][j]), int(d["agent"][j])))
    for lst in calls.values():
        lst.sort()
    n_calls = 0
    for i in range(q["sojourn"].size):
        e, arrive, soj, beta = int(q["env"][i]), int(q["arrive"][i]), int(q["sojourn"][i]), int(q["info"][i] & 0xFFFF)
        if len(starts[(e, arrive)]) != 1:                # two queries arrived in the same tick: the logs do not say which is which
            dirty[arrive:arrive + soj, e] = True
            continue
        lst = calls[(e, starts[(e, arrive)][0])]         # the table slot the query sat in; slots are reused over time
        s0 = lst.index((arrive, 0))
        mine = lst[s0:s0 + 3]
        assert [a for _, a in mine] == [0, 1, 2] and mine[2][0] < arrive + soj
        ends = [mine[1][0] - 1, mine[2][0] - 1, arrive + soj - 1]          # completion tick of each call
        for (t_issue, _), t_done in zip(mine, ends):
            ell = t_done + 1 - t_issue
            assert ell >= 1
            expect[t_done, e] += (ell << 16) // beta
            n_calls += 1
    # queries still in flight at the end have completed calls too: compare only the ticks before the oldest of them arrived
    got = np.rint(o.cost().astype(np.float64) * 65536.0).astype(np.int64)
    st = decode_state(o.state(), 2, spec.qcap, 4 * spec.qcap)
    n_cmp = 0
    for e in range(12):
        live_arrive = st["q_arrive"][e][st["q_live"][e] == 1]
        horizon = int(live_arrive.min()) if live_arrive.size else T
        ok = ~dirty[:horizon, e]
        assert np.array_equal(got[:horizon, e][ok], expect[:horizon, e][ok])
        n_cmp += int(ok.sum())
    assert n_cmp > 0.8 * 12 * T
    assert n_calls > 300 and got.sum() > 0


def test_single_call_constraint_violation_is_exactly_the_slo_miss(orc):
    """sum_k C_k <= 1 is the latency budget.  For a query with ONE call, l = sojourn, so the tick's
    Q16 cost exceeds 1.0 (65536) iff sojourn > budget iff the query is recorded as an SLO miss - an exact statement.
    Fails under: miss judged with >= instead of >; cost with the wrong denominator."""
    spec = tiny_spec(n_envs=8, N=1, n_ticks=600, qcap=32, rcap=96, rate_tick=0.02, slots=1, rates=[100], budget=(5, 60),
                     medians=(30, 60, 90))
    o = orc.Oracle(spec, seed=3)
    o.rollout(forced_single_blob(spec), 600)
    q = o.queries()
    got = np.rint(o.cost().astype(np.float64) * 65536.0).astype(np.int64)
    miss = o.miss().astype(np.int64)
    # keep ticks in which exactly one query finished and nothing was dropped
    fin_tick = q["arrive"] + q["sojourn"].astype(np.int64) - 1
    n = 0
    for i in range(q["sojourn"].size):
        e, t = int(q["env"][i]), int(fin_tick[i])
        if np.sum((q["env"] == e) & (fin_tick == t)) != 1:
            continue
        beta, soj = int(q["info"][i] & 0xFFFF), int(q["sojourn"][i])
        assert got[t, e] == (soj << 16) // beta
        assert (got[t, e] > 65536) == (soj > beta) == bool(miss[t, e])
        n += 1
    assert n > 40 and (miss.sum() > 5) and (miss.sum() < n)
    assert o.counters()[:, CN["dropped"]].sum() == 0


# --------------------------------------------------------------------------------- (b) success bit, R18 / R19
def _solve_rate(orc, topo, count, action, seed):
    spec = tiny_spec(n_envs=64, N=3, n_ticks=900, qcap=64, rcap=192, rate_tick=0.08, slots=64, rates=[150, 150, 150],
                     budget=(500, 500), medians=(20, 30, 40), seed=7)
    prob = np.array([[0.11, 0.27, 0.42], [0.58, 0.66, 0.81], [0.93, 0.35, 0.5]])     # p[model][depth], chosen here
    spec = spec.with_(succ_prob=prob, succ_thresh=np.floor(prob * 4294967296.0).astype(np.uint32))
    bias = np.full(9, -40.0)
    bias[action] = 40.0
    o = orc.Oracle(spec, seed=seed)
    o.rollout(planner_bias_blob(spec, topo=topo, count=count, exec_bias=bias), 900)
    q = o.queries()
    assert np.all(o.decisions(1)["payload"] == action)
    solved = ((q["info"] >> 16) & 1).astype(np.float64)
    return spec, solved


def test_success_bit_and_or_composition(orc):
    """R18: a call succeeds iff u32 draw < floor(p[m][d] 2^32); R19: a query is solved iff any of its calls succeeded.
    Every call is forced onto one (model, depth): single topology => solve rate = p within 4 sigma; debate with K = 3
    (two debaters + judge = 3 calls) => 1 - (1 - p)^3.  Fails under: >= instead of < in the success draw (rate 1 - p);
    AND instead of OR (p^3); only the last call counting (p)."""
    for action in (1, 5):                                  # (model 0, depth 1), (model 1, depth 2)
        spec, s1 = _solve_rate(orc, topo=0, count=1, action=action, seed=11)
        p = float(spec.succ_prob[action // 3][action % 3])
        assert p in (0.27, 0.81)
        assert s1.size > 3000
        assert abs(s1.mean() - p) < 4 * math.sqrt(p * (1 - p) / s1.size), (s1.mean(), p)
        _, s3 = _solve_rate(orc, topo=2, count=3, action=action, seed=12)
        p3 = 1 - (1 - p) ** 3
        assert s3.size > 3000
        assert abs(s3.mean() - p3) < 4 * math.sqrt(p3 * (1 - p3) / s3.size), (s3.mean(), p3)
        assert abs(s3.mean() - p) > 6 * math.sqrt(p * (1 - p) / s3.size)      # and it is not the single-call rate


# --------------------------------------------------------------------------------- (c) stage tables and K_eff, R17
def _stage_table(topo, K):
    """DESIGN.md R16/R17, typed independently: K_eff and the list of stages, each a list of agent ids."""
    if topo == 0:
        return 1, [[0]]
    if topo == 1:
        return K, [[a] for a in range(K)]
    keff = max(K, 2)
    if topo == 2:
        return keff, [list(range(keff - 1)), [keff - 1]]            # debaters in parallel, then the judge
    return keff, [[0], list(range(1, keff))]                        # writer, then the reviewers in parallel


def test_stage_tables_of_every_topology_and_count(orc):
    """R17: single [1]; chain [1]*K; debate [K-1 parallel, 1 judge]; review [1 writer, K-1 reviewers], K_eff =
    1 / K / max(K,2) / max(K,2); the next stage is dispatched the tick after the previous one completed.  With one
    fast uncontended model and frac = 0 the issue tick of every stage is a closed form of the calls' output tokens
    (recomputed from the Philox draw of each decision).  Fails under: debate as [1, K-1]; K_eff = K for debate with
    K = 1; the judge issued in the completion tick itself; reviewers issued one per tick."""
    for topo in range(4):
        for K in range(1, 5):
            keff, stages = _stage_table(topo, K)
            spec = tiny_spec(n_envs=8, N=1, n_ticks=400, qcap=64, rcap=192, rate_tick=0.02, slots=64, rates=[100],
                             budget=(2000, 2000), medians=(30, 70, 150), seed=1)
            o = orc.Oracle(spec, seed=100 + 4 * topo + K)
            o.rollout(planner_bias_blob(spec, topo=topo, count=K), 400)
            q, d = o.queries(), o.decisions(1)
            assert q["sojourn"].size > 15
            assert np.all(((q["info"] >> 17) & 3) == topo) and np.all(((q["info"] >> 19) & 7) == keff)
            by_q = {}
            for j in range(d["t"].size):
                env, t, qi, ag, a = int(d["env"][j]), int(d["t"][j]), int(d["q"][j]), int(d["agent"][j]), int(d["payload"][j])
                x = orc.philox(env, t, qi * 4 + ag, 0, (100 + 4 * topo + K), 4)       # key = (seed_lo, seed_hi ^ STREAM_EXEC)
                out = max(1, (int(spec.depth_median_tok[a % 3]) * int(spec.out_tok_mult_q16[x[1] >> 22])) >> 16)
                by_q.setdefault((env, qi), []).append((t, ag, math.ceil(out / 5.0)))   # 100 tok/s = 5 tok/tick, frac 0
            checked = 0
            for i in range(q["sojourn"].size):
                env, arrive, soj = int(q["env"][i]), int(q["arrive"][i]), int(q["sojourn"][i])
                # decisions of this query: those of a table slot of env within [arrive, arrive + sojourn)
                cands = [[c for c in lst if arrive <= c[0] < arrive + soj] for (e2, _), lst in by_q.items() if e2 == env]
                cands = [c for c in cands if c and min(x[0] for x in c) == arrive and len(c) == keff]
                match = 0
                for c in cands:
                    t_stage, ok = arrive, True
                    for st in stages:
                        calls = sorted(x for x in c if x[1] in st)
                        ok &= [x[1] for x in calls] == st and all(x[0] == t_stage for x in calls)
                        if not ok:
                            break
                        t_stage += max(x[2] for x in calls)        # all calls of the stage done, next stage the tick after
                    ok = ok and t_stage == arrive + soj
                    match += ok
                assert match >= 1, (topo, K, env, arrive, soj)
                checked += 1
            assert checked > 15


# --------------------------------------------------------------------------------- (d) head-of-line stop, R21
def test_kv_misfit_at_the_head_blocks_the_queue(orc):
    """R21 (vLLM-like): admission stops at the first request that does not fit, even if a later one would.  Input
    tokens are 60 or 900 (a two-valued table) against a KV capacity of 1000 with 8 slots, so that a 900-token head
    often meets a pool where only a 60-token request would fit.  From the state left by tick t-1: when a slot is
    free, the head (smallest (deadline, id) among WAITING) does not fit and some later request would, then at tick t
    nobody waiting behind that head may start.  Fails under: `continue` instead of `break` at the misfit."""
    tab = np.where(np.arange(1024) % 2 == 0, 60, 900).astype(np.uint32)
    spec = tiny_spec(n_envs=16, N=1, n_ticks=500, qcap=32, rcap=96, rate_tick=0.12, slots=8, rates=[100], kv_cap=1000,
                     budget=(50, 900), medians=(20, 40, 60), seed=2).with_(in_tok_table=tab)
    o = orc.Oracle(spec, seed=5)
    blob = forced_single_blob(spec)
    prev, blocked = None, 0
    for t in range(500):
        o.rollout(blob, 1)
        st = decode_state(o.state(), 1, spec.qcap, 4 * spec.qcap)
        if prev is not None:
            for e in range(16):
                w = np.nonzero(prev["r_state"][e] == ST_WAIT)[0]
                if len(w) < 2 or prev["n_run"][e, 0] >= 8:
                    continue
                keys = prev["r_deadline"][e][w].astype(np.int64) * 4096 + w
                order = w[np.argsort(keys)]
                need = (prev["r_in_tok"][e] + prev["r_out_total"][e] - prev["r_remaining"][e]).astype(np.int64)
                free = 1000 - int(prev["kv_used"][e, 0])
                head = order[0]
                if need[head] <= free or not np.any(need[order[1:]] <= free):
                    continue
                # new requests of tick t may only make the queue longer; the old head still does not fit
                behind = order[1:]
                assert st["r_state"][e][head] == ST_WAIT
                assert np.all(st["r_state"][e][behind] == ST_WAIT), (t, e)
                blocked += 1
        prev = st
    assert blocked > 20


# --------------------------------------------------------------------------------- (e) episodes, R33
def test_episode_boundary_is_a_hard_reset(orc):
    """R33: with episode_ticks = 50 every 50th tick has done = 1 and the env is emptied after it: no live query, no
    request, telemetry zero (EWMA included); live queries are counted as abandoned, and the query identity
    arrivals = finished + dropped + live + abandoned holds at every tick.  Fails under: done on tick % 50 == 0
    instead of (tick + 1) % 50 == 0; keeping the EWMA; not counting the abandoned queries."""
    spec = tiny_spec(n_envs=6, N=2, n_ticks=230, qcap=16, rcap=48, rate_tick=0.4, slots=2, budget=(30, 150), seed=5,
                     episode_ticks=50)
    blob = make_policy_blob(spec, seed=2)
    o = orc.Oracle(spec, seed=9)
    ab_prev = np.zeros(6, np.int64)
    for t in range(230):
        o.rollout(blob, 1)
        st = decode_state(o.state(), 2, spec.qcap, 4 * spec.qcap)
        c = o.counters().astype(np.int64)
        live = st["q_live"].sum(axis=1)
        assert np.array_equal(c[:, CN["arrivals"]], c[:, CN["finished"]] + c[:, CN["dropped"]] + live + c[:, CN["abandoned"]])
        boundary = (t + 1) % 50 == 0
        assert np.all(o.done()[0] == (1 if boundary else 0))
        if boundary:
            assert not o.state().any()                     # queries, requests, n_wait / n_run / kv_used / ewma: all zero
            assert np.all(c[:, CN["abandoned"]] >= ab_prev) and c[:, CN["abandoned"]].sum() > ab_prev.sum()
            ab_prev = c[:, CN["abandoned"]].copy()
        else:
            assert np.array_equal(c[:, CN["abandoned"]], ab_prev)
            if t % 50 > 10:
                assert st["q_live"].any() or st["ewma_q8"].any()
    # the tick after a boundary starts from an empty pool: its arrivals are the only live queries
    o2 = orc.Oracle(spec, seed=9)
    o2.rollout(blob, 51)
    st = decode_state(o2.state(), 2, spec.qcap, 4 * spec.qcap)
    assert np.all(st["q_arrive"][st["q_live"] == 1] == 50)


# --------------------------------------------------------------------------------- (f) near-boundary window, R25(3)
def test_near_boundary_window_is_one_millionth(orc):
    """R25(3) / north_star: a mismatching action is tolerated only if the uniform lies within 1e-6 of the CDF interval
    of that action.  Four equal logits => boundaries at 0.25, 0.5, 0.75.  Fails under: a window of 1e-5 or 1e-7; the
    interval of the neighbouring action; a missing division by Z."""
    _, _, cdf = orc.sample(np.full(4, 1.25, dtype=np.float32), 0.0)
    assert abs(float(cdf[-1]) - 4.0) < 1e-6                # running sums, not normalised: near_ok divides by Z
    for a, lo, hi in ((0, 0.0, 0.25), (1, 0.25, 0.5), (2, 0.5, 0.75), (3, 0.75, 1.0)):
        mid = 0.5 * (lo + hi)
        assert orc.near_ok(cdf, mid, a)
        for other in range(4):
            if other != a:
                assert not orc.near_ok(cdf, mid, other)
        if a < 3:                                          # just above the upper boundary of a
            assert orc.near_ok(cdf, float(np.float32(hi + 5e-7)), a)
            assert not orc.near_ok(cdf, float(np.float32(hi + 2e-6)), a)
        if a > 0:                                          # just below its lower boundary
            assert orc.near_ok(cdf, float(np.float32(lo - 5e-7)), a)
            assert not orc.near_ok(cdf, float(np.float32(lo - 2e-6)), a)
    # the first and the last action have no outer boundary
    assert orc.near_ok(cdf, 0.0, 0) and orc.near_ok(cdf, float(np.float32(1 - 2 ** -24)), 3)
