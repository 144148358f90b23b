"""im_gae_static - the returns kernel with its scratch in a static device array (no allocation) - against the existing
path (im_returns on a ctx).  Collected last on purpose (the suite runs with pytest -x).

The arithmetic of the walk is the same sequence of separately rounded fp32 operations (R31), so ADV / RET must equal
those of im_returns bit for bit, which is inside the 1e-5 relative tolerance tests/parity.py uses for returns; the cost
sum is a double added up in another order: 1e-12 relative.  Two calls in a row on DIFFERENT batches (the second one
smaller, so fewer CTAs than partial sums left in the scratch by the first; then the first again) show that what a call
leaves in the shared array does not leak into the next.
"""
import ctypes as C

import numpy as np
import pytest

from im_workload import make_policy_blob, make_pool_spec

pytestmark = pytest.mark.gpu

GAMMA, LAM, MU = 0.99, 0.95, 0.5


def _existing_path(n_envs, n_ticks, seed, episode_ticks=0):
    """Rollout + im_returns on a ctx; returns the ctx (kept alive: the tensors are views of its arena) and its arrays."""
    import torch
    from paper_2606_11440_b200 import (InfraMind, IM_TEL_ADV, IM_TEL_COST, IM_TEL_DONE, IM_TEL_RET, IM_TEL_REW, IM_TEL_VAL)
    spec = make_pool_spec(1, n_envs=n_envs, n_ticks=n_ticks)
    if episode_ticks:
        spec = spec.with_(episode_ticks=episode_ticks)
    g = InfraMind(spec, seed=seed, debug_flags=1)
    g.rollout(make_policy_blob(spec), n_ticks)
    g.returns(GAMMA, LAM, MU)
    g.sync()
    E, T = n_envs, n_ticks
    t = {name: g.device_tensor(what, dt).view(-1, E) for name, what, dt in (
        ("rew", IM_TEL_REW, torch.float32), ("cost", IM_TEL_COST, torch.float32), ("val", IM_TEL_VAL, torch.float32),
        ("done", IM_TEL_DONE, torch.uint8), ("adv", IM_TEL_ADV, torch.float32), ("ret", IM_TEL_RET, torch.float32))}
    assert t["rew"].shape == (T, E) and t["val"].shape == (T + 1, E)
    return g, t, float(g.sums()[0])


def _static_path(t):
    import torch
    from paper_2606_11440_b200 import gae_static
    adv, ret = torch.full_like(t["adv"], float("nan")), torch.full_like(t["ret"], float("nan"))
    s = torch.full((1,), float("nan"), dtype=torch.float64, device=adv.device)
    gae_static(t["rew"].contiguous(), t["cost"].contiguous(), t["val"].contiguous(), t["done"].contiguous(), adv, ret, s, GAMMA, LAM, MU)
    torch.cuda.synchronize()
    return adv, ret, float(s.item())


def _check(t, sum_cost_ref, out):
    import torch
    adv, ret, sum_cost = out
    for got, ref in ((adv, t["adv"]), (ret, t["ret"])):
        err = (got.double() - ref.double()).abs() / ref.double().abs().clamp(min=1.0)
        assert float(err.max()) <= 1e-5                       # the tolerance of tests/parity.py::compare_returns
        assert torch.equal(got, ref)                          # and in fact the same bits (same fp32 sequence)
    assert abs(sum_cost - sum_cost_ref) <= 1e-12 * max(1.0, abs(sum_cost_ref)), (sum_cost, sum_cost_ref)


def test_static_scratch_returns_equal_im_returns_on_two_calls_in_a_row():
    import torch
    ga, ta, sa = _existing_path(n_envs=3000, n_ticks=120, seed=5)                       # 12 CTAs, a ragged last one
    gb, tb, sb = _existing_path(n_envs=300, n_ticks=77, seed=6, episode_ticks=25)       # 2 CTAs, done rows inside
    assert sa > 0 and sb > 0 and tb["done"].any()
    _check(ta, sa, _static_path(ta))
    free0 = torch.cuda.mem_get_info()[0]
    _check(tb, sb, _static_path(tb))                  # right after: the scratch still holds the first call's 12 partial sums
    _check(ta, sa, _static_path(ta))
    first = _static_path(ta)
    assert first[2] == _static_path(ta)[2]            # fixed order of the sum: the same bits in every run
    assert torch.cuda.mem_get_info()[0] >= free0 - (8 << 20)      # nothing but torch's own small output tensors was taken
    ga.close(); gb.close()


def test_sizes_beyond_the_static_scratch_are_refused():
    import torch
    from paper_2606_11440_b200 import IM_GAE_STATIC_MAX_ENVS, load_library
    L = load_library()
    x = torch.zeros(16, dtype=torch.float32, device="cuda")
    err = C.create_string_buffer(512)
    p = x.data_ptr()                                  # never dereferenced: the size check comes first
    rc = L.im_gae_static(p, p, p, p, p, p, None, 4, IM_GAE_STATIC_MAX_ENVS + 1, GAMMA, LAM, MU, None, err, 512)
    assert rc == -6 and b"IM_GAE_STATIC_MAX_ENVS" in err.value
    assert L.im_gae_static(None, p, p, p, p, p, None, 4, 4, GAMMA, LAM, MU, None, err, 512) == -1
    assert L.im_gae_static(p, p, p, p, p, p, None, 0, 4, GAMMA, LAM, MU, None, err, 512) == -1
