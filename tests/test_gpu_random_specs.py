"""Randomised pool specs: the CUDA path against the oracle on small pools whose every knob is drawn at random
(number of models, slot counts 1..64 per model, table sizes, arrival levels, FCFS / EDF, KV preemption, cost mode,
episodes, prefill and input tokens, budgets, depth medians, the three policy kernels, ragged env counts, chunking).
The named cases of test_gpu_parity.py / test_gpu_edges.py pin what each of them is about; this sweep is there for the
combinations nobody thought of.  Seeds are fixed: a failure reproduces."""
import os

import numpy as np
import pytest

from helpers import tiny_spec
from test_gpu_parity import _run

pytestmark = pytest.mark.gpu


def _random_spec(case: int):
    rng = np.random.Generator(np.random.PCG64([case, 2606]))
    N = int(rng.integers(1, 17))
    # policy kernel: fp32 FFMA (any width that holds 3N+12 features), bf16 tcgen05 (64,128: zero-padded to the kernel's 256-wide hidden layers; 128,256)
    kinds = [("f32", 0, 64 if 3 * N + 12 > 32 else 32, int(rng.choice([16, 64])))]
    kinds.append(("mma", 1, 64, 128))
    kinds.append(("tc", 1, 128, 256))
    _, dtype, f_in, hidden = kinds[int(rng.integers(0, 3))]
    qcap = int(rng.choice([32, 64, 128]))
    preempt = int(rng.integers(0, 2))
    slots = rng.choice([1, 2, 3, 5, 8, 16, 33, 64], size=N).astype(np.uint32)
    medians = tuple(int(x) for x in np.sort(rng.integers(8, 400, size=3)))
    kv_cap = rng.integers(2 * medians[2] + 400, 6000, size=N).astype(np.uint32) if preempt else 32768
    lo = int(rng.integers(10, 120))
    hi = lo + int(rng.integers(1, 400))
    levels = rng.uniform(0.05, 2.5 if case % 3 == 0 else 1.0, size=int(rng.integers(1, 4)))   # every third case overloaded
    n_ticks = int(rng.integers(120, 260))
    spec = tiny_spec(n_envs=int(rng.integers(3, 100)), N=N, n_ticks=n_ticks, qcap=qcap, rcap=4 * qcap, rate_tick=levels,
                     dtype=dtype, f_in=f_in, hidden=hidden, sched_mode=int(rng.integers(0, 2)), kv_preempt=preempt,
                     kv_cap=kv_cap, slots=slots, seed=case, budget=(lo, hi), in_tok=int(rng.choice([0, 150])),
                     prefill=int(rng.choice([0, 700])), episode_ticks=int(rng.choice([0, 50, 97])),
                     cost_mode=int(rng.integers(0, 2)), medians=medians)
    # the logs are split into regions by env id: size them for the busiest env, not for the mean
    cap = (64 + spec.n_envs) * n_ticks * 48
    spec = spec.with_(log_cap_exec=cap, log_cap_plan=cap, log_cap_query=cap)
    # chunking of the rollout: a few cuts at random places (state persists across im_rollout calls)
    cuts = np.sort(rng.choice(np.arange(1, n_ticks), size=int(rng.integers(0, 4)), replace=False))
    chunks = [int(x) for x in np.diff(np.concatenate([[0], cuts, [n_ticks]]))]
    return spec, chunks, int(rng.integers(0, 1000))


@pytest.mark.parametrize("case", range(int(os.environ.get("IM_RANDOM_CASES", "48"))))   # more cases: a bug hunt, not the suite
def test_random_spec_parity(case):
    spec, chunks, seed = _random_spec(case)
    st = _run(spec, seed=seed, chunks=chunks)
    assert st["arrivals"] > 0
