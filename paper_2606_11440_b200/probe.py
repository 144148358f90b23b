"""ctypes binding of libimprobe.so (include/im_probe.h): the device's rate for accesses at data-dependent addresses.

Measurement only (bench.py's roofline of the tick simulation); argument marshalling, nothing else."""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libimprobe.so")
SHAPES = {"read16": 0, "write16": 1, "write32": 2, "rmw4": 3}
_lib = None


def load_probe():
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} missing: run `python -m paper_2606_11440_b200.build`")
        _lib = ctypes.CDLL(_SO)
        _lib.im_probe_random_access.restype = ctypes.c_int
        _lib.im_probe_random_access.argtypes = [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_size_t, ctypes.c_int, ctypes.c_uint32, ctypes.c_uint32,
                                                ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)]
    return _lib


def random_access_rates(device="cuda:0", gib=16, window_bytes=1 << 20, warps_per_sm=16, rounds=64):
    """{'read16': G accesses/s, ...} for every shape, on a scratch buffer of `gib` GiB that is freed afterwards."""
    import torch
    lib = load_probe()
    dev = torch.device(device)
    with torch.cuda.device(dev):
        buf = torch.empty(gib << 30, dtype=torch.uint8, device=dev)
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        n_threads = sms * warps_per_sm * 32 * 8                      # eight waves of resident warps
        out = {}
        for name, shape in SHAPES.items():
            g = ctypes.c_double(0.0)
            rc = lib.im_probe_random_access(buf.data_ptr(), buf.numel(), window_bytes, shape, n_threads, rounds,
                                            torch.cuda.current_stream().cuda_stream, ctypes.byref(g))
            if rc != 0:
                raise RuntimeError(f"im_probe_random_access({name}) failed: {rc}")
            out[name] = g.value
        del buf
        torch.cuda.empty_cache()
    return out
