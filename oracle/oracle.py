"""ctypes binding of the CPU oracle (oracle/inframind_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  It never imports the CUDA package and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "inframind_oracle.c")
_SO = os.path.join(_HERE, "build", "libinframind_oracle.so")

ORC_MAXN = 16
(ORC_REW, ORC_COST, ORC_VAL, ORC_DONE, ORC_MISS, ORC_ADV, ORC_RET, ORC_COUNTERS, ORC_SNAPSHOT, ORC_STATE,
 ORC_SCALARS, ORC_STATS) = range(1, 13)
COUNTER_NAMES = ["arrivals", "dropped", "finished", "solved", "missed", "calls_issued", "calls_done", "preemptions",
                 "sum_sojourn", "sum_live_mid", "plans", "exec_decisions", "sum_running", "sum_waiting",
                 "near_boundary", "abandoned"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no contraction, OpenMP for the timed mode)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        os.makedirs(os.path.dirname(_SO), exist_ok=True)
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
               "-Wall", "-o", _SO, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _SO


class _Model(C.Structure):
    _fields_ = [("rate_tok_s", C.c_uint32), ("slots", C.c_uint32), ("kv_cap", C.c_uint32),
                ("prefill_us_per_ktok", C.c_uint32), ("succ_thresh", C.c_uint32 * 3), ("kv_inv", C.c_float)]


class _Spec(C.Structure):
    _fields_ = [(n, C.c_uint32) for n in (
        "n_models", "qcap", "rcap", "max_ticks", "sched_mode", "kv_preempt", "cost_mode", "episode_ticks",
        "budget_norm_ticks", "n_levels", "policy_dtype", "f_in", "hidden", "in_tok_const", "mix_thresh", "keep_logits")]
    _fields_ += [("depth_median_tok", C.c_uint32 * 3), ("mix_lo", C.c_uint32 * 2), ("mix_hi", C.c_uint32 * 2),
                 ("model", _Model * ORC_MAXN),
                 ("out_tok_mult_q16", C.c_void_p), ("in_tok_table", C.c_void_p), ("arr_cdf", C.c_void_p)]


class _ForcedKind(C.Structure):
    _fields_ = [("off", C.c_void_p), ("t", C.c_void_p), ("q", C.c_void_p), ("agent", C.c_void_p),
                ("payload", C.c_void_p), ("logits", C.c_void_p)]


class _Forced(C.Structure):
    _fields_ = [("plan", _ForcedKind), ("exec", _ForcedKind)]


class _Ph4(C.Structure):
    _fields_ = [("v", C.c_uint32 * 4)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_philox4x32_10.restype = _Ph4
        L.orc_philox4x32_10.argtypes = [C.c_uint32] * 6
        L.orc_im_exp.restype = C.c_float
        L.orc_im_exp.argtypes = [C.c_float]
        L.orc_im_tanh.restype = C.c_float
        L.orc_im_tanh.argtypes = [C.c_float]
        L.orc_sample.restype = C.c_uint32
        L.orc_sample.argtypes = [C.c_void_p, C.c_uint32, C.c_float, C.c_void_p, C.c_void_p]
        L.orc_create.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_reset.argtypes = [C.c_void_p]
        L.orc_set_forced.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_rollout.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_int]
        L.orc_returns.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.orc_gae.argtypes = [C.c_void_p] * 4 + [C.c_uint32, C.c_uint32, C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_read.restype = C.c_int64
        L.orc_read.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_size_t]
        L.orc_state_words.restype = C.c_size_t
        L.orc_state_words.argtypes = [C.c_void_p]
        L.orc_log_count.restype = C.c_int64
        L.orc_log_count.argtypes = [C.c_void_p, C.c_int]
        L.orc_read_decisions.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 8
        L.orc_read_queries.argtypes = [C.c_void_p] * 5
        L.orc_queue_order.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_int32, C.c_void_p, C.c_uint32]
        L.orc_mlp_forward.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_near_ok.restype = C.c_int
        L.orc_near_ok.argtypes = [C.c_void_p, C.c_uint32, C.c_float, C.c_uint32]
        L.orc_tick.restype = C.c_int32
        L.orc_tick.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def philox(c0, c1, c2, c3, k0, k1):
    r = lib().orc_philox4x32_10(c0, c1, c2, c3, k0, k1)
    return [int(x) for x in r.v]


def im_exp(x: float) -> float:
    return float(lib().orc_im_exp(C.c_float(x)))


def im_tanh(x: float) -> float:
    return float(lib().orc_im_tanh(C.c_float(x)))


def sample(logits: np.ndarray, u: float):
    l = np.ascontiguousarray(logits, dtype=np.float32)
    lp = C.c_float()
    cdf = np.zeros(64, dtype=np.float32)
    a = lib().orc_sample(_p(l), l.size, C.c_float(u), C.byref(lp), _p(cdf))
    return int(a), float(lp.value), cdf[: l.size].copy()


def near_ok(cdf: np.ndarray, u: float, a: int) -> bool:
    """R25(3): is action `a` acceptable for uniform u, i.e. within 1e-6 of its CDF interval (cdf = running sums)."""
    c = np.ascontiguousarray(cdf, dtype=np.float32)
    return bool(lib().orc_near_ok(_p(c), c.size, C.c_float(u), a))


def gae(rew, cost, val, done, gamma, lam, mu):
    """Standalone R31 recurrence (float64) on [T][n] float32 arrays; val is [T+1][n]."""
    rew = np.ascontiguousarray(rew, dtype=np.float32)
    cost = np.ascontiguousarray(cost, dtype=np.float32)
    val = np.ascontiguousarray(val, dtype=np.float32)
    done = np.ascontiguousarray(done, dtype=np.uint8)
    T, n = rew.shape
    assert val.shape == (T + 1, n)
    adv = np.zeros((T, n), dtype=np.float64)
    ret = np.zeros((T, n), dtype=np.float64)
    lib().orc_gae(_p(rew), _p(cost), _p(val), _p(done), T, n, gamma, lam, mu, _p(adv), _p(ret))
    return adv, ret


class Oracle:
    """One oracle context over an explicit list of GLOBAL env ids (E-invariance, R2)."""

    def __init__(self, spec, seed: int = 0, env_ids: Optional[np.ndarray] = None, keep_logits: bool = False):
        L = lib()
        self.spec = spec
        if env_ids is None:
            env_ids = np.arange(spec.n_envs, dtype=np.uint32) + np.uint32(spec.env_id_base)
            levels = np.ascontiguousarray(spec.env_level, dtype=np.uint8)
        else:
            env_ids = np.ascontiguousarray(env_ids, dtype=np.uint32)
            levels = np.ascontiguousarray(spec.env_level[env_ids.astype(np.int64) - spec.env_id_base], dtype=np.uint8)
        self.env_ids = env_ids
        self.n = int(env_ids.size)
        self.N = spec.n_models
        s = _Spec()
        for name in ("n_models", "qcap", "rcap", "max_ticks", "sched_mode", "kv_preempt", "cost_mode", "episode_ticks",
                     "budget_norm_ticks", "n_levels", "policy_dtype", "f_in", "hidden", "in_tok_const", "mix_thresh"):
            setattr(s, name, int(getattr(spec, name)))
        s.keep_logits = 1 if keep_logits else 0
        self.keep_logits = keep_logits
        for i in range(3):
            s.depth_median_tok[i] = int(spec.depth_median_tok[i])
        for i in range(2):
            s.mix_lo[i] = int(spec.mix_lo[i])
            s.mix_hi[i] = int(spec.mix_hi[i])
        for k in range(spec.n_models):
            m = s.model[k]
            m.rate_tok_s = int(spec.rate_tok_s[k]); m.slots = int(spec.slots[k]); m.kv_cap = int(spec.kv_cap[k])
            m.prefill_us_per_ktok = int(spec.prefill_us_per_ktok[k]); m.kv_inv = float(spec.kv_inv[k])
            for d in range(3):
                m.succ_thresh[d] = int(spec.succ_thresh[k][d])
        self._keep = [np.ascontiguousarray(spec.out_tok_mult_q16, dtype=np.uint32),
                      None if spec.in_tok_table is None else np.ascontiguousarray(spec.in_tok_table, dtype=np.uint32),
                      np.ascontiguousarray(spec.arr_cdf, dtype=np.uint32)]
        s.out_tok_mult_q16 = self._keep[0].ctypes.data
        s.in_tok_table = None if self._keep[1] is None else self._keep[1].ctypes.data
        s.arr_cdf = self._keep[2].ctypes.data
        self._h = C.c_void_p()
        rc = L.orc_create(C.byref(s), self.n, _p(env_ids), _p(levels), C.c_uint64(seed), C.byref(self._h))
        if rc != 0:
            raise RuntimeError(f"orc_create failed: {rc}")
        self._forced_keep = None
        self.T = 0

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self):
        lib().orc_reset(self._h)

    @property
    def tick(self) -> int:
        return int(lib().orc_tick(self._h))

    def set_forced(self, plan: Optional[Dict[str, np.ndarray]] = None, exec_: Optional[Dict[str, np.ndarray]] = None):
        """Each dict: off[int64 n+1], t[int32], q[uint16], agent[uint8], payload[uint32], logits[float32 n x n_out] or None,
        sorted by (env_local, t, q, agent)."""
        if plan is None and exec_ is None:
            self._forced_keep = None
            lib().orc_set_forced(self._h, None)
            return
        f = _Forced()
        keep = []
        for dst, src in ((f.plan, plan), (f.exec, exec_)):
            if src is None:
                continue
            arrs = dict(off=np.ascontiguousarray(src["off"], dtype=np.int64), t=np.ascontiguousarray(src["t"], dtype=np.int32),
                        q=np.ascontiguousarray(src["q"], dtype=np.uint16), agent=np.ascontiguousarray(src["agent"], dtype=np.uint8),
                        payload=np.ascontiguousarray(src["payload"], dtype=np.uint32))
            lg = src.get("logits")
            if lg is not None:
                arrs["logits"] = np.ascontiguousarray(lg, dtype=np.float32)
            for k, v in arrs.items():
                setattr(dst, k, v.ctypes.data)
            keep.append(arrs)
        self._forced_keep = (f, keep)
        lib().orc_set_forced(self._h, C.byref(f))

    def rollout(self, blob: np.ndarray, n_ticks: int, n_threads: int = 1):
        blob = np.ascontiguousarray(blob, dtype=np.uint8)
        rc = lib().orc_rollout(self._h, _p(blob), n_ticks, n_threads)
        if rc != 0:
            raise RuntimeError(f"orc_rollout failed: {rc}")
        self.T = n_ticks

    def returns(self, gamma: float, lam: float, mu: float):
        rc = lib().orc_returns(self._h, gamma, lam, mu)
        if rc != 0:
            raise RuntimeError(f"orc_returns failed: {rc}")

    def _read(self, what, dtype, shape):
        out = np.zeros(shape, dtype=dtype)
        rc = lib().orc_read(self._h, what, _p(out), out.nbytes)
        if rc < 0:
            raise RuntimeError(f"orc_read({what}) failed: {rc}")
        assert rc == out.nbytes, (rc, out.nbytes)
        return out

    def rew(self): return self._read(ORC_REW, np.float32, (self.T, self.n))
    def cost(self): return self._read(ORC_COST, np.float32, (self.T, self.n))
    def val(self): return self._read(ORC_VAL, np.float32, (self.T + 1, self.n))
    def done(self): return self._read(ORC_DONE, np.uint8, (self.T, self.n))
    def miss(self): return self._read(ORC_MISS, np.uint8, (self.T, self.n))
    def adv(self): return self._read(ORC_ADV, np.float64, (self.T, self.n))
    def ret(self): return self._read(ORC_RET, np.float64, (self.T, self.n))
    def counters(self): return self._read(ORC_COUNTERS, np.uint64, (self.n, 16))
    def snapshot(self): return self._read(ORC_SNAPSHOT, np.uint32, (self.n, self.N, 4))
    def state(self): return self._read(ORC_STATE, np.uint32, (self.n, int(lib().orc_state_words(self._h))))

    def scalars(self):
        v = self._read(ORC_SCALARS, np.float64, (5,))
        return dict(cbar=v[0], ubar=v[1], usigma=v[2], sum_cost=v[3], n_final=int(v[4]))

    def stats(self):
        v = self._read(ORC_STATS, np.float64, (5,))
        return dict(desync=int(v[0]), hard=int(v[1]), near=int(v[2]), max_logit_diff=float(v[3]), max_value_diff=float(v[4]))

    def decisions(self, kind: int):
        """kind 0 = planner, 1 = executor. Arrays sorted by (env_local, t, q, agent)."""
        n = int(lib().orc_log_count(self._h, kind))
        n_out = 3 * self.N + 1 if kind else 24
        d = dict(env_local=np.zeros(n, np.uint32), t=np.zeros(n, np.int32), q=np.zeros(n, np.uint16),
                 agent=np.zeros(n, np.uint8), payload=np.zeros(n, np.uint32), logp=np.zeros(n, np.float32),
                 value=np.zeros(n, np.float32))
        lg = np.zeros((n, n_out), np.float32) if self.keep_logits else None
        lib().orc_read_decisions(self._h, kind, _p(d["env_local"]), _p(d["t"]), _p(d["q"]), _p(d["agent"]),
                                 _p(d["payload"]), _p(d["logp"]), _p(d["value"]), _p(lg))
        d["logits"] = lg
        d["env"] = self.env_ids[d["env_local"].astype(np.int64)] if n else np.zeros(0, np.uint32)
        return d

    def queries(self):
        n = int(lib().orc_log_count(self._h, 2))
        d = dict(env=np.zeros(n, np.uint32), arrive=np.zeros(n, np.int32), sojourn=np.zeros(n, np.uint32),
                 info=np.zeros(n, np.uint32))
        lib().orc_read_queries(self._h, _p(d["env"]), _p(d["arrive"]), _p(d["sojourn"]), _p(d["info"]))
        return d

    def queue_order(self, env_local: int, model: int, t: int):
        buf = np.zeros(self.spec.rcap, np.uint32)
        n = lib().orc_queue_order(self._h, env_local, model, t, _p(buf), buf.size)
        return buf[:n].copy()

    def mlp_forward(self, which: int, x: np.ndarray):
        """Run the currently loaded policy (after a rollout) on one feature vector."""
        x = np.ascontiguousarray(x, dtype=np.float32)
        out = np.zeros(64, np.float32)
        lib().orc_mlp_forward(self._h, which, _p(x), _p(out))
        return out[: (3 * self.N + 1 if which else 24)].copy()
