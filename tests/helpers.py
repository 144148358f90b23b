"""Test-side helpers: decode the canonical STATE dump (include/inframind.h, IM_TEL_STATE) and build small specs.

The dump layout is part of the ABI contract, typed here a third time (independently of both the oracle
and the CUDA path) so that tests can check invariants from raw words.
"""
from __future__ import annotations

import numpy as np

from im_workload import make_pool_spec, poisson_cdf_row
from im_workload.workload import PoolSpec, pack_policy_blob, lognormal_table

ST_FREE, ST_WAIT, ST_RUN = 0, 1, 2


def decode_state(words: np.ndarray, N: int, qcap: int, rcap: int):
    """words: [n_envs][4N + 4*qcap + 5*rcap] u32 -> dict of arrays; rcap = 4*qcap, request row = query*4 + agent."""
    w = np.asarray(words, dtype=np.uint32)
    n = w.shape[0]
    m = w[:, : 4 * N].reshape(n, N, 4)
    q = w[:, 4 * N: 4 * N + 4 * qcap].reshape(n, qcap, 4)
    r = w[:, 4 * N + 4 * qcap:].reshape(n, rcap, 5)
    q0 = q[:, :, 0]
    r0 = r[:, :, 0]
    return dict(
        n_wait=m[:, :, 0], n_run=m[:, :, 1], kv_used=m[:, :, 2], ewma_q8=m[:, :, 3],
        q_live=(q0 & 1), q_planned=(q0 >> 1) & 1, q_topo=(q0 >> 2) & 3, q_cnt=(q0 >> 4) & 3, q_keff=(q0 >> 6) & 7,
        q_stage=(q0 >> 9) & 7, q_nstages=(q0 >> 12) & 7, q_pending=(q0 >> 15) & 3, q_succ=(q0 >> 17) & 1,
        q_roles=(q0 >> 18) & 0xFF, q_deadline=q[:, :, 1].astype(np.int32), q_arrive=q[:, :, 2].astype(np.int32),
        q_budget=q[:, :, 3] & 0xFFFF, q_in_tok=q[:, :, 3] >> 16,
        r_state=r0 & 3, r_model=(r0 >> 2) & 15, r_depth=(r0 >> 6) & 3, r_agent=(r0 >> 8) & 3, r_succ=(r0 >> 10) & 1,
        r_query=r0 >> 16, r_deadline=r[:, :, 1].astype(np.int32), r_issue=r[:, :, 2].astype(np.int32),
        r_remaining=r[:, :, 3] & 0xFFFF, r_slot1=r[:, :, 3] >> 16, r_out_total=r[:, :, 4] & 0xFFFF,
        r_in_tok=r[:, :, 4] >> 16,
    )


def tiny_spec(n_envs=4, N=2, n_ticks=64, qcap=16, rcap=48, rate_tick=0.3, dtype=0, f_in=32, hidden=16,
              sched_mode=1, kv_preempt=0, kv_cap=32768, slots=2, rates=None, seed=0, budget=(40, 200),
              in_tok=0, prefill=0, episode_ticks=0, cost_mode=0, medians=(16, 48, 96)) -> PoolSpec:
    """A small hand-sized pool for pins; every field explicit."""
    rng = np.random.Generator(np.random.PCG64([seed, 99]))
    rates = np.asarray(rates if rates is not None else rng.integers(40, 201, size=N), dtype=np.uint32)
    p = np.median(rng.random(size=(N, 3, 3)), axis=2)
    kv = np.full(N, kv_cap, dtype=np.uint32) if np.isscalar(kv_cap) else np.asarray(kv_cap, dtype=np.uint32)
    sl = np.full(N, slots, dtype=np.uint32) if np.isscalar(slots) else np.asarray(slots, dtype=np.uint32)
    rate_rows = np.atleast_1d(np.asarray(rate_tick, dtype=np.float64))
    return PoolSpec(
        config_id=0, n_envs=n_envs, n_ticks=n_ticks, n_models=N, qcap=qcap, rcap=rcap, max_ticks=n_ticks,
        sched_mode=sched_mode, kv_preempt=kv_preempt, cost_mode=cost_mode, episode_ticks=episode_ticks,
        budget_norm_ticks=max(budget[1], 1), n_levels=len(rate_rows), policy_dtype=dtype, f_in=f_in, hidden=hidden,
        debug_flags=0, in_tok_const=in_tok, depth_median_tok=np.asarray(medians, dtype=np.uint32),
        mix_thresh=0xFFFFFFFF, mix_lo=np.array([budget[0]] * 2, dtype=np.uint32), mix_hi=np.array([budget[1]] * 2, dtype=np.uint32),
        rate_tok_s=rates, slots=sl, kv_cap=kv, prefill_us_per_ktok=np.full(N, prefill, dtype=np.uint32),
        succ_thresh=np.floor(p * 4294967296.0).astype(np.uint32), kv_inv=(1.0 / kv.astype(np.float64)).astype(np.float32),
        out_tok_mult_q16=lognormal_table(1.0, 0.4, scale=65536.0), in_tok_table=None,
        arr_cdf=np.stack([poisson_cdf_row(float(m)) for m in rate_rows]).astype(np.uint32),
        env_level=(np.arange(n_envs) % len(rate_rows)).astype(np.uint8),
        log_cap_exec=n_envs * n_ticks * 40 + 1024, log_cap_plan=n_envs * n_ticks * 32 + 1024,
        log_cap_query=n_envs * n_ticks * 32 + 1024,
        arr_rate_tick=rate_rows, succ_prob=p,
    )


def forced_single_blob(spec: PoolSpec, exec_bias=None, seed=0) -> np.ndarray:
    """Policy whose planner always picks topology 'single' (W3=0, bias +40) and whose executor is uniform
    (or follows exec_bias logits): used by the M/M/1 and stamp pins."""
    H, F, N = spec.hidden, spec.f_in, spec.n_models
    z = lambda *s: np.zeros(s, dtype=np.float32)
    b3 = z(24)
    b3[0] = 40.0   # topology single
    b3[4] = 40.0   # count 1
    eb = z(3 * N + 1)
    if exec_bias is not None:
        eb[: 3 * N] = np.asarray(exec_bias, dtype=np.float32)
    arrays = dict(plan_W1=z(H, F), plan_b1=z(H), plan_W2=z(H, H), plan_b2=z(H), plan_W3=z(24, H), plan_b3=b3,
                  exec_W1=z(H, F), exec_b1=z(H), exec_W2=z(H, H), exec_b2=z(H), exec_W3=z(3 * N + 1, H), exec_b3=eb)
    return pack_policy_blob(spec.policy_dtype, F, H, N, arrays)


def planner_bias_blob(spec: PoolSpec, topo: int, count: int, exec_bias=None) -> np.ndarray:
    """Policy forcing a given topology and agent count (biases +-40), zero weights elsewhere."""
    H, F, N = spec.hidden, spec.f_in, spec.n_models
    z = lambda *s: np.zeros(s, dtype=np.float32)
    b3 = z(24)
    b3[topo] = 40.0
    b3[4 + count - 1] = 40.0
    eb = z(3 * N + 1)
    if exec_bias is not None:
        eb[: 3 * N] = np.asarray(exec_bias, dtype=np.float32)
    arrays = dict(plan_W1=z(H, F), plan_b1=z(H), plan_W2=z(H, H), plan_b2=z(H), plan_W3=z(24, H), plan_b3=b3,
                  exec_W1=z(H, F), exec_b1=z(H), exec_W2=z(H, H), exec_b2=z(H), exec_W3=z(3 * N + 1, H), exec_b3=eb)
    return pack_policy_blob(spec.policy_dtype, F, H, N, arrays)
