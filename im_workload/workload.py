"""Synthetic workloads for the INFRAMIND CMDP rollout (BASELINE.json configs[0..4]).

Everything here is *input generation*: pool parameters, integer distribution tables, arrival
levels and random policy weights.  The recipe is stated in DESIGN.md ("Input recipe") and
follows SURVEY.md §8(d).  Nothing here implements Philox, the tick, the MLP or GAE.

The paper itself measures on five public benchmarks served by five
LLMs under vLLM with max_num_seqs=16, Poisson arrivals and budget tiers 10..300 s; none of
that is available here, so these seeded synthetic pools stand in for it.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, Optional

import numpy as np

DT_US = 50_000  # one tick = 50 ms (BASELINE.json north_star)
TICKS_PER_S = 20

# nominal tokens per query used to convert utilisation -> arrival rate:
# 2.25 calls (uniform planner) x mean(128,512,1536) x exp(0.4^2/2)
TOK_PER_QUERY_NOMINAL = 2.25 * (128 + 512 + 1536) / 3.0 * math.exp(0.08)

BLOB_MAGIC = 0x494D5042  # 'IMPB'


@dataclass
class PoolSpec:
    """Plain-data description of one pool + workload (all dynamics parameters are integers)."""
    config_id: int
    n_envs: int
    n_ticks: int                      # the config's rollout length T (not part of the C spec)
    n_models: int
    qcap: int
    rcap: int
    max_ticks: int
    sched_mode: int                   # 0 FCFS, 1 EDF
    kv_preempt: int
    cost_mode: int                    # 0: sum l/beta, 1: SLO-miss count
    episode_ticks: int
    budget_norm_ticks: int
    n_levels: int
    policy_dtype: int                 # 0 fp32, 1 bf16
    f_in: int
    hidden: int
    debug_flags: int
    in_tok_const: int
    depth_median_tok: np.ndarray      # [3] u32
    mix_thresh: int                   # component 0 iff x < mix_thresh
    mix_lo: np.ndarray                # [2] u32 ticks
    mix_hi: np.ndarray                # [2] u32 ticks
    rate_tok_s: np.ndarray            # [N] u32
    slots: np.ndarray                 # [N] u32
    kv_cap: np.ndarray                # [N] u32
    prefill_us_per_ktok: np.ndarray   # [N] u32
    succ_thresh: np.ndarray           # [N][3] u32 = floor(p * 2^32)
    kv_inv: np.ndarray                # [N] f32 = fp32(1/kv_cap)
    out_tok_mult_q16: np.ndarray      # [1024] u32
    in_tok_table: Optional[np.ndarray]  # [1024] u32 or None
    arr_cdf: np.ndarray               # [n_levels][32] u32
    env_level: np.ndarray             # [n_envs] u8
    env_id_base: int = 0              # global id of env 0 (multi-GPU shards)
    log_cap_exec: int = 0             # decision-log capacities (rows); 0 => sized by library
    log_cap_plan: int = 0
    log_cap_query: int = 0
    gamma: float = 0.99
    lam_gae: float = 0.95
    mu_lag: float = 0.5
    arr_rate_tick: np.ndarray = field(default_factory=lambda: np.zeros(1))  # [n_levels] float64 (info only)
    succ_prob: np.ndarray = field(default_factory=lambda: np.zeros((1, 3)))  # [N][3] float64 (info only)

    def with_(self, **kw) -> "PoolSpec":
        return replace(self, **kw)

    def subset(self, env_ids: np.ndarray) -> "PoolSpec":
        """Spec for a subset of envs (same pool rows); callers pass env ids explicitly to the oracle."""
        env_ids = np.asarray(env_ids, dtype=np.int64)
        return replace(self, n_envs=int(env_ids.size), env_level=self.env_level[env_ids].copy())


# ----------------------------------------------------------------------------------------------
# distribution tables (float64 -> integer once, here, so both sides receive identical bytes)
# ----------------------------------------------------------------------------------------------

def poisson_cdf_row(mean_per_tick: float) -> np.ndarray:
    """32 u32 thresholds: row[j] = floor(P(X<=j) * 2^32) for j<31, row[31] = 2^32-1 (unused pad).

    The count drawn from a u32 x is #{j < 31 : x >= row[j]} (0..31)."""
    row = np.empty(32, dtype=np.uint64)
    term = math.exp(-mean_per_tick)
    cdf = 0.0
    for j in range(31):
        cdf += term
        row[j] = min(int(math.floor(min(cdf, 1.0) * 4294967296.0)), 0xFFFFFFFF)
        term *= mean_per_tick / (j + 1)
    row[31] = 0xFFFFFFFF
    # enforce monotonicity against float round-off
    for j in range(1, 32):
        if row[j] < row[j - 1]:
            row[j] = row[j - 1]
    return row.astype(np.uint32)


def _ndtri(p: np.ndarray) -> np.ndarray:
    from scipy.special import ndtri
    return ndtri(p)


def lognormal_table(median: float, sigma: float, scale: float = 1.0, n: int = 1024) -> np.ndarray:
    """n-entry quantile table of median*exp(sigma*Phi^-1((i+1/2)/n)) * scale, rounded to u32."""
    q = (np.arange(n, dtype=np.float64) + 0.5) / n
    v = median * np.exp(sigma * _ndtri(q)) * scale
    return np.rint(v).astype(np.uint32)


def exponential_table_q16(n: int = 1024) -> np.ndarray:
    """Q16 multipliers with exponential(1) quantiles -ln(1-(i+1/2)/n) (M/M/1 pin)."""
    q = (np.arange(n, dtype=np.float64) + 0.5) / n
    return np.rint(-np.log1p(-q) * 65536.0).astype(np.uint32)


# ----------------------------------------------------------------------------------------------
# configs
# ----------------------------------------------------------------------------------------------

CONFIGS: Dict[int, dict] = {
    1: dict(E=64, N=5, T=200, dtype=0, f_in=32, hidden=64, qcap=256, rcap=768),
    2: dict(E=4096, N=5, T=2000, dtype=0, f_in=32, hidden=64, qcap=256, rcap=768),
    # chunk: ticks per im_rollout call (trajectory / log capacity); the 4000-tick rollouts of configs 3-4 run as
    # 8 consecutive calls of 500 ticks with persistent env state, so that the logs of one call fit in HBM
    3: dict(E=65536, N=8, T=4000, dtype=1, f_in=64, hidden=128, qcap=256, rcap=768, chunk=500),
    4: dict(E=131072, N=16, T=4000, dtype=1, f_in=128, hidden=256, qcap=512, rcap=1536, chunk=500),
    5: dict(E=262144, N=16, T=512, dtype=1, f_in=128, hidden=256, qcap=512, rcap=1536),
}


def make_pool_spec(config_id: int, seed: int = 0, n_envs: Optional[int] = None,
                   n_ticks: Optional[int] = None, debug_flags: int = 0, max_ticks: Optional[int] = None) -> PoolSpec:
    """Materialise BASELINE.json configs[config_id-1] from `seed`.

    n_envs / n_ticks override E / T for parity tests on a slice; pool rows depend only on
    (config_id, seed), env levels only on (config_id, seed, env id) for the *full* E of the config
    (so env e of a slice equals env e of the full run: E-invariance).
    """
    cfg = CONFIGS[config_id]
    E_full, N, T = cfg["E"], cfg["N"], cfg["T"]
    E = E_full if n_envs is None else int(n_envs)
    T = T if n_ticks is None else int(n_ticks)
    chunk = min(T, int(max_ticks) if max_ticks is not None else cfg.get("chunk", T))
    rng = np.random.Generator(np.random.PCG64([config_id, seed, 0x1F2A]))

    if config_id in (1, 2):
        rate = rng.integers(40, 201, size=N)
        slots = np.full(N, 16)
        kv = np.full(N, 32768)
        kv_preempt = 0
        prefill = np.zeros(N, dtype=np.int64)
    else:
        rate = rng.integers(20, 301, size=N)
        slots = 8 << rng.integers(0, 4, size=N)
        kv = 16384 << rng.integers(0, 4, size=N)
        kv_preempt = 1
        prefill = rng.integers(200, 2001, size=N) if config_id >= 4 else np.zeros(N, dtype=np.int64)

    # success probabilities: median of three uniforms is exactly Beta(2,2)
    p = np.median(rng.random(size=(N, 3, 3)), axis=2)
    succ_thresh = np.minimum(np.floor(p * 4294967296.0), 4294967295.0).astype(np.uint32)

    # budgets (ticks) — SURVEY R7
    if config_id == 5:
        mix_thresh = 0x80000000
        mix_lo = np.array([100, 800], dtype=np.uint32)
        mix_hi = np.array([300, 2400], dtype=np.uint32)
        budget_norm = 2400
    else:
        mix_thresh = 0xFFFFFFFF
        mix_lo = np.array([200, 200], dtype=np.uint32)
        mix_hi = np.array([1200, 1200], dtype=np.uint32)
        budget_norm = 1200

    # arrival levels — SURVEY R6
    cap_tok_s = float(np.sum(slots * rate))
    if config_id == 1:
        rates_tick = np.array([2.0 / TICKS_PER_S])
    elif config_id == 2:
        rho = np.linspace(0.3, 0.9, 64)
        rates_tick = rho * cap_tok_s / TOK_PER_QUERY_NOMINAL / TICKS_PER_S
    elif config_id == 3:
        rates_tick = np.array([1.2 * cap_tok_s / TOK_PER_QUERY_NOMINAL / TICKS_PER_S])
    else:
        rho = np.linspace(0.2, 1.3, 64)
        rates_tick = rho * cap_tok_s / TOK_PER_QUERY_NOMINAL / TICKS_PER_S
    n_levels = len(rates_tick)
    arr_cdf = np.stack([poisson_cdf_row(float(m)) for m in rates_tick]).astype(np.uint32)

    ids = np.arange(E, dtype=np.int64)
    if config_id == 2:
        # level random per env, a pure function of (seed, env id)
        lv_rng = np.random.Generator(np.random.PCG64([config_id, seed, 0x77]))
        env_level = lv_rng.integers(0, n_levels, size=E_full).astype(np.uint8)[:E] if E <= E_full \
            else lv_rng.integers(0, n_levels, size=E).astype(np.uint8)
    elif config_id in (4, 5):
        env_level = ((ids % E_full) * n_levels // E_full).astype(np.uint8)
    else:
        env_level = np.zeros(E, dtype=np.uint8)

    in_tok_table = lognormal_table(800.0, 0.6) if config_id >= 4 else None

    mean_rate = float(np.mean(rates_tick[env_level.astype(np.int64)])) if E > 0 else 0.0
    exec_nom = E * chunk * mean_rate * 2.25
    plan_nom = E * chunk * mean_rate
    spec = PoolSpec(
        config_id=config_id, n_envs=E, n_ticks=T, n_models=N,
        qcap=cfg["qcap"], rcap=cfg["rcap"], max_ticks=chunk,
        sched_mode=1, kv_preempt=kv_preempt, cost_mode=0, episode_ticks=0,
        budget_norm_ticks=budget_norm, n_levels=n_levels,
        policy_dtype=cfg["dtype"], f_in=cfg["f_in"], hidden=cfg["hidden"],
        debug_flags=debug_flags, in_tok_const=0,
        depth_median_tok=np.array([128, 512, 1536], dtype=np.uint32),
        mix_thresh=mix_thresh, mix_lo=mix_lo, mix_hi=mix_hi,
        rate_tok_s=rate.astype(np.uint32), slots=slots.astype(np.uint32), kv_cap=kv.astype(np.uint32),
        prefill_us_per_ktok=prefill.astype(np.uint32), succ_thresh=succ_thresh,
        kv_inv=(1.0 / kv.astype(np.float64)).astype(np.float32),
        out_tok_mult_q16=lognormal_table(1.0, 0.4, scale=65536.0),
        in_tok_table=in_tok_table, arr_cdf=arr_cdf, env_level=env_level,
        log_cap_exec=int(exec_nom * 1.4) + 64 * E + 4096,
        log_cap_plan=int(plan_nom * 1.3) + 32 * E + 4096,
        log_cap_query=int(plan_nom * 1.3) + 32 * E + 4096,
        arr_rate_tick=np.asarray(rates_tick, dtype=np.float64), succ_prob=p,
    )
    return spec


# ----------------------------------------------------------------------------------------------
# policy weights (SURVEY R26 blob)
# ----------------------------------------------------------------------------------------------

def _f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16 bit patterns (u16)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    r = ((u >> 16) & 1) + 0x7FFF
    return ((u + r) >> 16).astype(np.uint16)


def _bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << 16).view(np.float32)


def _layout(dtype: int, f_in: int, hidden: int, n_models: int):
    """[(name, shape, is_weight)] in blob order."""
    out = []
    for net, n_out in (("plan", 24), ("exec", 3 * n_models + 1)):
        out += [(f"{net}_W1", (hidden, f_in), True), (f"{net}_b1", (hidden,), False),
                (f"{net}_W2", (hidden, hidden), True), (f"{net}_b2", (hidden,), False),
                (f"{net}_W3", (n_out, hidden), True), (f"{net}_b3", (n_out,), False)]
    return out


def pack_policy_blob(dtype: int, f_in: int, hidden: int, n_models: int, arrays: Dict[str, np.ndarray]) -> np.ndarray:
    """Pack fp32 arrays into the blob (weights rounded to bf16 when dtype==1; biases stay fp32)."""
    parts = [np.array([BLOB_MAGIC, dtype, f_in, hidden, 24, 3 * n_models + 1, n_models, 0], dtype=np.uint32).tobytes()]
    for name, shape, is_w in _layout(dtype, f_in, hidden, n_models):
        a = np.ascontiguousarray(arrays[name], dtype=np.float32).reshape(shape)
        raw = _f32_to_bf16_bits(a).tobytes() if (is_w and dtype == 1) else a.tobytes()
        pad = (-len(raw)) % 16
        parts.append(raw + b"\0" * pad)
    return np.frombuffer(b"".join(parts), dtype=np.uint8).copy()


def blob_views(blob: np.ndarray) -> Dict[str, np.ndarray]:
    """Decode a blob back to fp32 arrays (bf16 weights widened exactly)."""
    hdr = blob[:32].view(np.uint32)
    assert int(hdr[0]) == BLOB_MAGIC
    dtype, f_in, hidden, n_models = int(hdr[1]), int(hdr[2]), int(hdr[3]), int(hdr[6])
    out = {"dtype": dtype, "f_in": f_in, "hidden": hidden, "n_models": n_models}
    off = 32
    for name, shape, is_w in _layout(dtype, f_in, hidden, n_models):
        n = int(np.prod(shape))
        if is_w and dtype == 1:
            a = _bf16_bits_to_f32(blob[off:off + 2 * n].view(np.uint16)).reshape(shape)
            nbytes = 2 * n
        else:
            a = blob[off:off + 4 * n].view(np.float32).reshape(shape)
            nbytes = 4 * n
        out[name] = a.copy()
        off += nbytes + ((-nbytes) % 16)
    assert off == blob.size
    return out


def make_policy_blob(spec: PoolSpec, seed: int = 0, scale: float = 1.0) -> np.ndarray:
    """Random policy: U(-1/sqrt(fan_in), 1/sqrt(fan_in)) * scale for weights and biases."""
    rng = np.random.Generator(np.random.PCG64([0xB10B, seed, spec.f_in, spec.hidden, spec.n_models]))
    arrays = {}
    for name, shape, is_w in _layout(spec.policy_dtype, spec.f_in, spec.hidden, spec.n_models):
        fan_in = shape[-1] if is_w else {"1": spec.f_in, "2": spec.hidden, "3": spec.hidden}[name[-1]]
        bound = scale / math.sqrt(fan_in)
        arrays[name] = rng.uniform(-bound, bound, size=shape).astype(np.float32)
    return pack_policy_blob(spec.policy_dtype, spec.f_in, spec.hidden, spec.n_models, arrays)
