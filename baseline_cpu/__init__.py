"""Stronger CPU baseline - a reporting baseline for bench.py only.

``baseline_cpu/dedisp_cpu_vec.cpp``: threaded, time-blocked, compiler-vectorised brute force (the modern
counterpart of the paper's SSE/AVX kernel). Not the oracle (that stays plain and untuned) and
not reachable from the product: only ``bench.py`` and ``tests/test_cpu_baseline.py`` import this package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_cpu_vec.cpp")
_lib = None


def _cpu_tag() -> str:
    """-march=native code must not travel between machines: one library per CPU feature set."""
    import hashlib
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


_LIB = os.path.join(_HERE, f"libdedisp_cpu_vec_{_cpu_tag()}.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["g++", "-O3", "-march=native", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
                        "-o", _LIB, _SRC], check=True)
    return _LIB


def dedisperse(nchans, fch1, foff, tsamp, dm_list, data: np.ndarray, nsamp_out: int, nthreads: int | None = None) -> np.ndarray:
    """All DM rows of ``dm_list`` from ``data[nchans][nsamp_in]`` (uint8 -> int32, float32 -> float32)."""
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    assert data.ndim == 2 and data.shape[0] == nchans and data.flags.c_contiguous and data.dtype in (np.uint8, np.float32)
    out = np.empty((dm.size, nsamp_out), dtype=np.int32 if data.dtype == np.uint8 else np.float32)
    fn = _lib.cpu_vec_dedisperse_u8 if data.dtype == np.uint8 else _lib.cpu_vec_dedisperse_f32
    fn.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p,
                   ctypes.c_longlong, ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_int]
    rc = fn(nchans, fch1, foff, tsamp, dm.ctypes.data, dm.size, data.ctypes.data, data.shape[1], data.shape[1], nsamp_out,
            out.ctypes.data, int(nthreads or os.cpu_count() or 1))
    if rc:
        raise ValueError(f"cpu_vec_dedisperse rc={rc}")
    return out
