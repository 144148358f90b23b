"""CPU-side checks of the C-ABI library (no compute calls without a GPU): it loads, exports every symbol that
include/inframind.h declares, validates specs on the host, and sizes arenas."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from im_workload import make_pool_spec

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_11440_b200 import build
    build.build()
    from paper_2606_11440_b200 import load_library
    return load_library()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "inframind.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(im_[a-z_]+)\s*\(", hdr))
    assert {"im_create", "im_reset", "im_rollout", "im_returns", "im_read_telemetry"} <= declared   # the north star's five
    for name in declared:
        assert hasattr(lib, name), name
    from paper_2606_11440_b200 import EXPORTS
    assert set(EXPORTS) == declared


def test_probe_library_exports_its_symbol(lib):
    """include/im_probe.h (the measurement probe of bench.py) is a library of its own; a bad argument is refused on the host."""
    from paper_2606_11440_b200.probe import load_probe
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "im_probe.h")).read(), flags=re.S)
    declared = set(re.findall(r"\b(im_[a-z_]+)\s*\(", hdr))
    assert declared == {"im_probe_random_access"}
    p = load_probe()
    for name in declared:
        assert hasattr(p, name)
        assert not hasattr(lib, name)                       # the boundary of the method holds nothing but the method
    g = C.c_double(0.0)
    assert p.im_probe_random_access(None, 1 << 30, 1 << 20, 0, 64, 1, None, C.byref(g)) == -1


def test_spec_struct_layout_matches_header(lib):
    """The ctypes mirror must have the C struct's size: 26 u32 + 3 u64 + 16 models x 32 B + 4 pointers."""
    from paper_2606_11440_b200.binding import im_pool_spec, im_model_spec
    assert C.sizeof(im_model_spec) == 32
    assert C.sizeof(im_pool_spec) == 26 * 4 + 3 * 8 + 16 * 32 + 4 * 8


def test_create_validates_on_host(lib):
    from paper_2606_11440_b200 import marshal_spec
    spec = make_pool_spec(1, n_envs=16, n_ticks=10)
    cs, keep = marshal_spec(spec)
    h = C.c_void_p()
    assert lib.im_create(C.byref(cs), 16, C.c_uint64(0), C.byref(h)) == 0
    assert lib.im_launch_count(h) == 0
    # compute calls before im_bind are state errors, not crashes
    assert lib.im_reset(h) == -5
    assert lib.im_rollout(h, C.c_void_p(keep[0].ctypes.data), 1) == -5
    assert lib.im_returns(h, 0.99, 0.95, 0.5) == -5
    assert b"im_bind" in lib.im_last_error(h) or b"rollout" in lib.im_last_error(h)
    lib.im_destroy(h)
    for field, value, code in (("n_models", 17, -2), ("rcap", 700, -2), ("qcap", 300, -2), ("abi_version", 9, -2),
                               ("max_ticks", 9000, -2), ("f_in", 8, -2), ("n_levels", 0, -2)):
        cs2, keep2 = marshal_spec(spec)
        setattr(cs2, field, value)
        h2 = C.c_void_p()
        assert lib.im_create(C.byref(cs2), 16, C.c_uint64(0), C.byref(h2)) == code, field
        assert h2.value is None and len(lib.im_last_error(None)) > 0
    cs3, keep3 = marshal_spec(spec)
    bad = keep3[2].copy()
    bad[0, 5] = 0                                       # non-monotone CDF row
    cs3.arr_cdf = bad.ctypes.data
    assert lib.im_create(C.byref(cs3), 16, C.c_uint64(0), C.byref(C.c_void_p())) == -2
    assert lib.im_create(None, 16, C.c_uint64(0), C.byref(C.c_void_p())) == -1
    assert lib.im_create(C.byref(cs), 0, C.c_uint64(0), C.byref(C.c_void_p())) == -1


def test_arena_sizes_fit_the_b200(lib):
    """All five configs fit 180 GB of HBM3e with the logs the bench keeps."""
    from paper_2606_11440_b200 import marshal_spec
    sizes = {}
    for cfg in (1, 2, 3, 5):
        spec = make_pool_spec(cfg)
        cs, keep = marshal_spec(spec, debug_flags=1)
        sizes[cfg] = lib.im_arena_bytes(C.byref(cs), spec.n_envs)
        assert 0 < sizes[cfg] < 170e9, (cfg, sizes[cfg])
    assert sizes[1] < sizes[2] < sizes[3]
    # state bytes/env within 2x of SURVEY §8's estimate (19.6 KB cfg1-3, 39.2 KB cfg4-5)
    spec = make_pool_spec(5, n_envs=1024, n_ticks=1)
    cs, keep = marshal_spec(spec.with_(log_cap_exec=64, log_cap_plan=64, log_cap_query=64), debug_flags=0)
    per_env = lib.im_arena_bytes(C.byref(cs), 1024) / 1024
    assert 39_000 < per_env < 80_000, per_env
