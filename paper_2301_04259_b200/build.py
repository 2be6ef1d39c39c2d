"""In-tree build of the C-ABI shared library (sm_100a only).

``python -m paper_2301_04259_b200.build`` or ``build()``: one nvcc invocation, no JIT cache - the
resulting ``libsoap_b200.so`` sits next to this file so that it travels with the source tree.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsoap_b200.so")
SOURCES = [os.path.join(CSRC, "soap_api.cu")]
HEADERS = [os.path.join(CSRC, f) for f in ("ptx_helpers.cuh", "composite.cuh", "contrast.cuh", "geometry.cuh", "active.cuh", "sia.cuh", "sia_f32.cuh", "lsf.cuh", "rv.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "soap_b200.h")]
# measurement aids of bench.py (the FP32 rate probe): a library of their own, never loaded by the product
BENCH_LIB = os.path.join(HERE, "libsoap_b200_bench.so")
BENCH_SOURCES = [os.path.join(CSRC, "bench_probe.cu")]
BENCH_HEADERS = [os.path.join(CSRC, f) for f in ("ptx_helpers.cuh", "probe.cuh")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "--use_fast_math=false",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(lib, deps) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(f) > t for f in deps if os.path.exists(f))


def needs_build() -> bool:
    return _stale(LIB, SOURCES + HEADERS)


def _compile(lib, sources, verbose) -> None:
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")] + os.environ.get("SOAP_NVCC_EXTRA", "").split()
    cmd = [_nvcc()] + flags + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + sources
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed building {os.path.basename(lib)}")


def build(force: bool = False, verbose: bool = False) -> str:
    """Builds libsoap_b200.so (the product) and libsoap_b200_bench.so (bench.py's probe); returns the product's path."""
    if force or needs_build():
        _compile(LIB, SOURCES, verbose)
    if force or _stale(BENCH_LIB, BENCH_SOURCES + BENCH_HEADERS):
        _compile(BENCH_LIB, BENCH_SOURCES, verbose)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
