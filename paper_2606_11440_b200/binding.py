"""Thin ctypes binding of libinframind.so (include/inframind.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  PyTorch lends the device arena (one
uint8 tensor) and the CUDA stream; nothing here computes.  There is no CPU fallback: if the shared library
is missing, or no sm_100 device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libinframind.so")

IM_MAX_MODELS = 16
IM_ABI_VERSION = 1
IM_FLAG_LOG_DECISIONS, IM_FLAG_LOG_LOGITS = 1, 2
(IM_TEL_SNAPSHOT, IM_TEL_COUNTERS, IM_TEL_REW, IM_TEL_COST, IM_TEL_VAL, IM_TEL_DONE, IM_TEL_MISS, IM_TEL_ADV, IM_TEL_RET,
 IM_TEL_SCALARS, IM_TEL_DECISIONS_EXEC, IM_TEL_DECISIONS_PLAN, IM_TEL_QUERIES, IM_TEL_UNORM, IM_TEL_STATE,
 IM_TEL_QUEUE_ORDER, IM_TEL_TABLES, IM_TEL_LOGITS_EXEC, IM_TEL_LOGITS_PLAN, IM_TEL_SUMS) = range(1, 21)

EXPORTS = ["im_arena_bytes", "im_create", "im_bind", "im_reset", "im_rollout", "im_returns", "im_returns_finish", "im_read_telemetry",
           "im_device_ptr", "im_launch_count", "im_set_profiling", "im_kernel_times", "im_destroy", "im_last_error", "im_gae_static"]
IM_GAE_STATIC_MAX_ENVS = 1048576


class im_model_spec(C.Structure):
    _fields_ = [("rate_tok_s", C.c_uint32), ("slots", C.c_uint32), ("kv_cap", C.c_uint32),
                ("prefill_us_per_ktok", C.c_uint32), ("succ_thresh", C.c_uint32 * 3), ("kv_inv", C.c_float)]


class im_pool_spec(C.Structure):
    _fields_ = [(n, C.c_uint32) for n in (
        "abi_version", "n_models", "qcap", "rcap", "max_ticks", "sched_mode", "kv_preempt", "cost_mode", "episode_ticks",
        "budget_norm_ticks", "n_levels", "policy_dtype", "f_in", "hidden", "debug_flags", "in_tok_const", "mix_thresh",
        "env_id_base")]
    _fields_ += [("depth_median_tok", C.c_uint32 * 3), ("mix_lo", C.c_uint32 * 2), ("mix_hi", C.c_uint32 * 2),
                 ("reserved", C.c_uint32),
                 ("log_cap_exec", C.c_uint64), ("log_cap_plan", C.c_uint64), ("log_cap_query", C.c_uint64),
                 ("model", im_model_spec * IM_MAX_MODELS),
                 ("out_tok_mult_q16", C.c_void_p), ("in_tok_table", C.c_void_p), ("arr_cdf", C.c_void_p),
                 ("env_level", C.c_void_p)]


_lib = None


def load_library():
    """Load libinframind.so; raises (no fallback) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: run `python -m paper_2606_11440_b200.build` (no CPU fallback exists)")
        L = C.CDLL(_SO)
        L.im_arena_bytes.restype = C.c_size_t
        L.im_arena_bytes.argtypes = [C.c_void_p, C.c_uint32]
        L.im_create.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_void_p]
        L.im_bind.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.im_reset.argtypes = [C.c_void_p]
        L.im_rollout.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32]
        L.im_returns.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_float]
        L.im_returns_finish.argtypes = [C.c_void_p, C.c_void_p]
        L.im_read_telemetry.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_size_t, C.c_void_p]
        L.im_device_ptr.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]
        L.im_launch_count.restype = C.c_uint64
        L.im_launch_count.argtypes = [C.c_void_p]
        L.im_set_profiling.argtypes = [C.c_void_p, C.c_int]
        L.im_kernel_times.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.im_destroy.restype = None
        L.im_destroy.argtypes = [C.c_void_p]
        L.im_last_error.restype = C.c_char_p
        L.im_last_error.argtypes = [C.c_void_p]
        L.im_gae_static.argtypes = [C.c_void_p] * 7 + [C.c_uint32, C.c_uint32, C.c_float, C.c_float, C.c_float, C.c_void_p, C.c_char_p, C.c_size_t]
        _lib = L
    return _lib


def gae_static(rew, cost, val, done, adv, ret, sum_cost, gamma: float, lam: float, mu: float, stream=None):
    """im_gae_static: GAE / Lagrangian returns on the caller's CUDA tensors, no ctx and no allocation (static scratch inside
    the library, <= IM_GAE_STATIC_MAX_ENVS envs).  rew / cost [T, E] f32, val [T + 1, E] f32, done [T, E] u8, adv / ret
    [T, E] f32 (written), sum_cost: one-element f64 CUDA tensor (written) or None.  Argument marshalling only."""
    import torch
    T, E = rew.shape
    for x, dt, sh in ((rew, torch.float32, (T, E)), (cost, torch.float32, (T, E)), (val, torch.float32, (T + 1, E)),
                      (done, torch.uint8, (T, E)), (adv, torch.float32, (T, E)), (ret, torch.float32, (T, E))):
        assert x.is_cuda and x.is_contiguous() and x.dtype == dt and tuple(x.shape) == sh
    assert sum_cost is None or (sum_cost.is_cuda and sum_cost.dtype == torch.float64 and sum_cost.numel() == 1)
    err = C.create_string_buffer(512)
    st = (stream if stream is not None else torch.cuda.current_stream(rew.device)).cuda_stream
    with torch.cuda.device(rew.device):
        rc = load_library().im_gae_static(rew.data_ptr(), cost.data_ptr(), val.data_ptr(), done.data_ptr(), adv.data_ptr(), ret.data_ptr(),
                                          None if sum_cost is None else sum_cost.data_ptr(), T, E, gamma, lam, mu, st, err, 512)
    if rc != 0:
        raise IMError(rc, err.value.decode())


def marshal_spec(spec, debug_flags: Optional[int] = None):
    """PoolSpec (im_workload) -> (im_pool_spec, keep-alive list)."""
    s = im_pool_spec()
    s.abi_version = IM_ABI_VERSION
    for name in ("n_models", "qcap", "rcap", "max_ticks", "sched_mode", "kv_preempt", "cost_mode", "episode_ticks",
                 "budget_norm_ticks", "n_levels", "policy_dtype", "f_in", "hidden", "in_tok_const", "mix_thresh", "env_id_base"):
        setattr(s, name, int(getattr(spec, name)))
    s.debug_flags = int(spec.debug_flags if debug_flags is None else debug_flags)
    for i in range(3):
        s.depth_median_tok[i] = int(spec.depth_median_tok[i])
    for i in range(2):
        s.mix_lo[i] = int(spec.mix_lo[i])
        s.mix_hi[i] = int(spec.mix_hi[i])
    s.log_cap_exec, s.log_cap_plan, s.log_cap_query = int(spec.log_cap_exec), int(spec.log_cap_plan), int(spec.log_cap_query)
    for k in range(spec.n_models):
        m = s.model[k]
        m.rate_tok_s, m.slots, m.kv_cap = int(spec.rate_tok_s[k]), int(spec.slots[k]), int(spec.kv_cap[k])
        m.prefill_us_per_ktok, m.kv_inv = int(spec.prefill_us_per_ktok[k]), float(spec.kv_inv[k])
        for d in range(3):
            m.succ_thresh[d] = int(spec.succ_thresh[k][d])
    keep = [np.ascontiguousarray(spec.out_tok_mult_q16, dtype=np.uint32),
            None if spec.in_tok_table is None else np.ascontiguousarray(spec.in_tok_table, dtype=np.uint32),
            np.ascontiguousarray(spec.arr_cdf, dtype=np.uint32), np.ascontiguousarray(spec.env_level, dtype=np.uint8)]
    s.out_tok_mult_q16 = keep[0].ctypes.data
    s.in_tok_table = None if keep[1] is None else keep[1].ctypes.data
    s.arr_cdf = keep[2].ctypes.data
    s.env_level = keep[3].ctypes.data
    return s, keep


class IMError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libinframind error {code}: {msg}")
        self.code = code


class InfraMind:
    """im_create + im_bind on a torch-owned arena; methods mirror the C ABI one to one."""

    def __init__(self, spec, seed: int = 0, device: str = "cuda:0", debug_flags: Optional[int] = None, stream=None,
                 arena=None):
        import torch
        self._L = load_library()
        self.spec = spec
        self.E, self.N = int(spec.n_envs), int(spec.n_models)
        cs, self._keep = marshal_spec(spec, debug_flags)
        self._cspec = cs
        self._h = C.c_void_p()
        rc = self._L.im_create(C.byref(cs), self.E, C.c_uint64(seed), C.byref(self._h))
        if rc != 0:
            raise IMError(rc, self._L.im_last_error(None).decode())
        nbytes = int(self._L.im_arena_bytes(C.byref(cs), self.E))
        if not torch.cuda.is_available():
            self._L.im_destroy(self._h)
            self._h = None
            raise RuntimeError("no CUDA device: libinframind has no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        # `arena` lets several contexts of the SAME spec (e.g. one per seed) share one allocation, used one at a time
        self.arena = arena if arena is not None else torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        assert self.arena.numel() >= nbytes + 256
        ptr = (self.arena.data_ptr() + 255) & ~255
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._check(self._L.im_bind(self._h, C.c_void_p(ptr), nbytes, C.c_void_p(self.stream.cuda_stream)))
        self.arena_bytes = nbytes
        self.T = 0

    def _check(self, rc: int):
        if rc != 0:
            raise IMError(rc, self._L.im_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.im_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the five calls of the north star
    def reset(self):
        self._check(self._L.im_reset(self._h))

    def rollout(self, policy_weights, n_ticks: int):
        """policy_weights: numpy uint8 blob (host) or a torch CUDA uint8 tensor (device)."""
        if isinstance(policy_weights, np.ndarray):
            blob = np.ascontiguousarray(policy_weights, dtype=np.uint8)
            self._blob_keep = blob
            ptr = blob.ctypes.data
        else:
            self._blob_keep = policy_weights
            ptr = policy_weights.data_ptr()
        self._check(self._L.im_rollout(self._h, C.c_void_p(ptr), int(n_ticks)))
        self.T = int(n_ticks)

    def returns(self, gamma: float, lam: float, mu: float):
        self._check(self._L.im_returns(self._h, gamma, lam, mu))

    def sums(self) -> np.ndarray:
        """IM_TEL_SUMS: float64 [sum_cost, n_final, sum_U, sum_U2] of this ctx (what an env-sharded job all-reduces)."""
        return self.read(IM_TEL_SUMS, np.float64, (4,))

    def returns_finish(self, global_sums):
        """im_returns_finish: re-normalise UNORM / SCALARS with the job-wide sums (host array of 4 doubles)."""
        g = np.ascontiguousarray(global_sums, dtype=np.float64)
        assert g.shape == (4,)
        self._check(self._L.im_returns_finish(self._h, g.ctypes.data_as(C.c_void_p)))

    def read(self, what: int, dtype, shape=None, out: Optional[np.ndarray] = None) -> np.ndarray:
        """im_read_telemetry into a numpy array (size queried first when shape is None)."""
        written = C.c_size_t()
        if out is None:
            if shape is None:
                self._check(self._L.im_read_telemetry(self._h, what, None, 0, C.byref(written)))
                n = written.value // np.dtype(dtype).itemsize
                out = np.zeros(n, dtype=dtype)
            else:
                out = np.zeros(shape, dtype=dtype)
        self._check(self._L.im_read_telemetry(self._h, what, out.ctypes.data_as(C.c_void_p), out.nbytes, C.byref(written)))
        assert written.value == out.nbytes, (written.value, out.nbytes)
        return out

    def read_into(self, what: int, host_tensor) -> int:
        """im_read_telemetry into a (pinned) torch CPU tensor; returns bytes written."""
        written = C.c_size_t()
        self._check(self._L.im_read_telemetry(self._h, what, C.c_void_p(host_tensor.data_ptr()),
                                              host_tensor.numel() * host_tensor.element_size(), C.byref(written)))
        return int(written.value)

    # ---- convenience views of im_read_telemetry
    def rew(self): return self.read(IM_TEL_REW, np.float32, (self.T, self.E))
    def cost(self): return self.read(IM_TEL_COST, np.float32, (self.T, self.E))
    def val(self): return self.read(IM_TEL_VAL, np.float32, (self.T + 1, self.E))
    def done(self): return self.read(IM_TEL_DONE, np.uint8, (self.T, self.E))
    def miss(self): return self.read(IM_TEL_MISS, np.uint8, (self.T, self.E))
    def adv(self): return self.read(IM_TEL_ADV, np.float32, (self.T, self.E))
    def ret(self): return self.read(IM_TEL_RET, np.float32, (self.T, self.E))
    def counters(self): return self.read(IM_TEL_COUNTERS, np.uint64, (self.E, 16))
    def snapshot(self): return self.read(IM_TEL_SNAPSHOT, np.uint32, (self.E, self.N, 4))
    def state(self): return self.read(IM_TEL_STATE, np.uint32, (self.E, 4 * self.N + 4 * self.spec.qcap + 20 * self.spec.qcap))
    def queue_order(self): return self.read(IM_TEL_QUEUE_ORDER, np.uint32, (self.E, self.N + 1 + self.spec.rcap))

    def scalars(self):
        v = self.read(IM_TEL_SCALARS, np.float64, (8,))
        return dict(cbar=v[0], ubar=v[1], usigma=v[2], sum_cost=v[3], n_final=int(v[4]), n_exec=int(v[5]), n_plan=int(v[6]), tick=int(v[7]))

    def decisions(self, kind: int, logits: bool = False):
        """kind 0 planner, 1 executor -> dict of arrays in log (unsorted) order."""
        raw = self.read(IM_TEL_DECISIONS_EXEC if kind else IM_TEL_DECISIONS_PLAN, np.uint32).reshape(-1, 6)
        d = dict(env=raw[:, 0].copy(), t=raw[:, 1].astype(np.int32), q=(raw[:, 2] & 0xFFFF).astype(np.uint16),
                 agent=(raw[:, 2] >> 16).astype(np.uint8), payload=raw[:, 3].copy(),
                 logp=raw[:, 4].copy().view(np.float32), value=raw[:, 5].copy().view(np.float32))
        if logits:
            n_out = 3 * self.N + 1 if kind else 24
            d["logits"] = self.read(IM_TEL_LOGITS_EXEC if kind else IM_TEL_LOGITS_PLAN, np.float32).reshape(-1, n_out)
        return d

    def queries(self, unorm: bool = False):
        raw = self.read(IM_TEL_QUERIES, np.uint32).reshape(-1, 4)
        d = dict(env=raw[:, 0].copy(), arrive=raw[:, 1].astype(np.int32), sojourn=raw[:, 2].copy(), info=raw[:, 3].copy())
        if unorm:
            d["unorm"] = self.read(IM_TEL_UNORM, np.float32)
        return d

    def device_tensor(self, what: int, dtype):
        """Zero-copy torch view of a trajectory array inside the arena (im_device_ptr)."""
        import torch
        p, b = C.c_void_p(), C.c_size_t()
        self._check(self._L.im_device_ptr(self._h, what, C.byref(p), C.byref(b)))
        base = (self.arena.data_ptr() + 255) & ~255
        off = p.value - base + (base - self.arena.data_ptr())
        return self.arena[off: off + b.value].view(dtype)

    def set_profiling(self, on: bool):
        self._check(self._L.im_set_profiling(self._h, 1 if on else 0))

    def kernel_times(self):
        """{'sim': (ms, launches), 'plan': ..., 'exec': ..., 'returns': ..., 'serve': ...} since the last call."""
        ms = (C.c_double * 5)()
        n = (C.c_uint64 * 5)()
        self._check(self._L.im_kernel_times(self._h, ms, n))
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(("sim", "plan", "exec", "returns", "serve"))}

    @property
    def launches(self) -> int:
        return int(self._L.im_launch_count(self._h))

    def sync(self):
        self.stream.synchronize()
