"""Lock-step parity protocol between the CUDA path (through the C ABI) and the CPU oracle.

GPU runs with LOG_DECISIONS (+LOG_LOGITS for bf16).  The oracle replays the same global env ids chunk by
chunk, consuming the GPU's decision log sorted by (env, tick, query, agent): fp32 policies are recomputed
by the oracle and must give the same action (R22-R24); bf16 policies are teacher-forced (R25).  After every
chunk the full integer state, trajectories and counters are compared exactly.
"""
from __future__ import annotations

import numpy as np

from oracle import oracle as O


def forced_from_gpu(dec, env_ids: np.ndarray, with_logits: bool):
    """GPU decision dict -> oracle forced dict restricted to env_ids (sorted unique global ids)."""
    env_ids = np.asarray(env_ids, dtype=np.uint32)
    pos = np.searchsorted(env_ids, dec["env"])
    pos = np.minimum(pos, env_ids.size - 1)
    keep = env_ids[pos] == dec["env"]
    idx = np.nonzero(keep)[0]
    loc = pos[idx].astype(np.int64)
    order = np.lexsort((dec["agent"][idx], dec["q"][idx], dec["t"][idx], loc))
    idx, loc = idx[order], loc[order]
    off = np.searchsorted(loc, np.arange(env_ids.size + 1)).astype(np.int64)
    out = dict(off=off, t=dec["t"][idx], q=dec["q"][idx], agent=dec["agent"][idx], payload=dec["payload"][idx],
               logp=dec["logp"][idx], value=dec["value"][idx], env_local=loc)
    if with_logits:
        out["logits"] = np.ascontiguousarray(dec["logits"][idx])
    return out


def compare_chunk(gpu, orc, env_ids, n_ticks, blob, bf16: bool, stats: dict, check_state=True):
    """Advance both sides by n_ticks and compare. `gpu` is an InfraMind, `orc` an Oracle over env_ids."""
    base = int(gpu.spec.env_id_base)
    cols = (np.asarray(env_ids, dtype=np.int64) - base)
    gpu.rollout(blob, n_ticks)
    gd_exec = gpu.decisions(1, logits=bf16)
    gd_plan = gpu.decisions(0, logits=bf16)
    f_exec = forced_from_gpu(gd_exec, env_ids, bf16)
    f_plan = forced_from_gpu(gd_plan, env_ids, bf16)
    orc.set_forced(plan=f_plan, exec_=f_exec)
    orc.rollout(blob, n_ticks, n_threads=8)
    od_exec, od_plan = orc.decisions(1), orc.decisions(0)
    # decisions: same multiset in canonical order, same actions
    for name, f, o in (("exec", f_exec, od_exec), ("plan", f_plan, od_plan)):
        assert f["t"].size == o["t"].size, f"{name}: decision count {f['t'].size} vs oracle {o['t'].size}"
        assert np.array_equal(f["env_local"], o["env_local"].astype(np.int64)), name
        assert np.array_equal(f["t"], o["t"]) and np.array_equal(f["q"], o["q"]) and np.array_equal(f["agent"], o["agent"]), name
        assert np.array_equal(f["payload"], o["payload"]), f"{name}: actions differ"
        if f["t"].size:
            stats["max_logp_diff"] = max(stats.get("max_logp_diff", 0.0), float(np.max(np.abs(f["logp"] - o["logp"]))))
    if f_exec["t"].size:
        dv = np.abs(f_exec["value"].astype(np.float64) - od_exec["value"])
        stats["max_dec_value_diff"] = max(stats.get("max_dec_value_diff", 0.0), float(dv.max()))
    stats["decisions"] = stats.get("decisions", 0) + int(f_exec["t"].size + f_plan["t"].size)
    # trajectories
    for name in ("rew", "cost", "miss", "done"):
        g, o = getattr(gpu, name)()[:, cols], getattr(orc, name)()
        assert np.array_equal(g, o), f"{name} differs"
    gv, ov = gpu.val()[:, cols], orc.val()
    if bf16:
        stats["max_val_diff"] = max(stats.get("max_val_diff", 0.0), float(np.max(np.abs(gv - ov))))
    else:
        assert np.array_equal(gv, ov), "critic values differ (fp32 contract is bit-exact)"
    gc, oc = gpu.counters()[cols], orc.counters()
    oc[:, 14] = 0
    if not np.array_equal(gc, oc):
        bad = np.argwhere(gc != oc)
        raise AssertionError(f"counters differ at (env_col, counter) {bad[:8].tolist()}: gpu {gc[gc != oc][:8].tolist()} oracle {oc[gc != oc][:8].tolist()}")
    if check_state:
        gs = gpu.state()[cols]
        os_ = orc.state()
        if not np.array_equal(gs, os_):
            bad = np.argwhere(gs != os_)
            raise AssertionError(f"state differs at (env_col, word) {bad[:8].tolist()} of {len(bad)}")
    return gd_exec, gd_plan


def finish_stats(orc, stats, bf16):
    s = orc.stats()
    assert s["desync"] == 0, s
    assert s["hard"] == 0, s
    n = max(stats.get("decisions", 0), 1)
    assert s["near"] / n < 1e-5 or s["near"] == 0, s
    assert stats.get("max_logp_diff", 0.0) <= 1e-5, stats
    if bf16:
        assert s["max_logit_diff"] <= 2e-2 and s["max_value_diff"] <= 2e-2, s
        assert stats.get("max_val_diff", 0.0) <= 2e-2, stats
    else:
        assert stats.get("max_dec_value_diff", 0.0) == 0.0, stats
    stats.update(s)
    return stats


def compare_returns(gpu, orc, env_ids, gamma, lam, mu, bf16, whole_batch=True):
    """GAE / utility / C-bar parity (R31, R32). bf16: the oracle recurrence is fed the GPU's arrays."""
    base = int(gpu.spec.env_id_base)
    cols = (np.asarray(env_ids, dtype=np.int64) - base)
    gpu.returns(gamma, lam, mu)
    g_adv, g_ret = gpu.adv()[:, cols], gpu.ret()[:, cols]
    if bf16:
        o_adv, o_ret = O.gae(gpu.rew()[:, cols], gpu.cost()[:, cols], gpu.val()[:, cols], gpu.done()[:, cols], gamma, lam, mu)
    else:
        orc.returns(gamma, lam, mu)
        o_adv, o_ret = orc.adv(), orc.ret()
    for g, o in ((g_adv, o_adv), (g_ret, o_ret)):
        err = np.abs(g.astype(np.float64) - o) / np.maximum(1.0, np.abs(o))
        assert err.max() <= 1e-5, err.max()
    if whole_batch:
        orc.returns(gamma, lam, mu)
        so, sg = orc.scalars(), gpu.scalars()
        assert so["n_final"] == sg["n_final"]
        for k in ("cbar", "ubar", "usigma"):
            assert abs(so[k] - sg[k]) <= 1e-5 * max(1.0, abs(so[k])), (k, so[k], sg[k])
        gq = gpu.queries(unorm=True)
        U = ((gq["info"] >> 16) & 1).astype(np.float64) - mu * gq["sojourn"].astype(np.float64) / (gq["info"] & 0xFFFF)
        z = (U - so["ubar"]) / (so["usigma"] + 1e-8)
        if U.size:
            assert np.max(np.abs(gq["unorm"] - z)) <= 1e-5 * max(1.0, np.max(np.abs(z))) + 2e-5
        # query logs agree as multisets
        oq = orc.queries()
        a = np.stack([gq["env"], gq["arrive"].astype(np.uint32), gq["sojourn"], gq["info"]], 1)
        b = np.stack([oq["env"], oq["arrive"].astype(np.uint32), oq["sojourn"], oq["info"]], 1)
        a = a[np.lexsort(a.T[::-1])]; b = b[np.lexsort(b.T[::-1])]
        assert np.array_equal(a, b), "query logs differ"
