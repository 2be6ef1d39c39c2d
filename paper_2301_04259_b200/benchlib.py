"""Loader of libsoap_b200_bench.so: measurement aids for bench.py (csrc/bench_probe.cu).  Not part of the product ABI; the
package does not import this module."""
from __future__ import annotations

import ctypes
import os

_LIB = None


def load() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        from . import build as _build
        path = _build.BENCH_LIB
        if not os.path.exists(path):
            _build.build()
        _LIB = ctypes.CDLL(path)
        _LIB.soap_bench_fp32_rate.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        _LIB.soap_bench_fp32_rate.restype = ctypes.c_int
    return _LIB


def fp32_rate(device: int = 0, packed: bool = True) -> float:
    """FP32 FMAs per second of `device`: FFMA2 (packed) or FFMA chains, best of four repetitions."""
    out = ctypes.c_double(0.0)
    rc = load().soap_bench_fp32_rate(int(device), 1 if packed else 0, ctypes.byref(out))
    if rc != 0:
        raise RuntimeError(f"soap_bench_fp32_rate failed: cudaError {rc}")
    return float(out.value)
