"""ORACLE — test infrastructure, NOT the product.

ctypes loader for ``oracle/dedisp_oracle.cpp``, the plain single-threaded CPU
statement of brute-force incoherent de-dispersion (§2; formula from
BASELINE.json:north_star). Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package. It imports nothing from ``paper_1111_6399_b200``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_dedisp.so")
_SRC_CT = os.path.join(_HERE, "corner_turn_oracle.cpp")
_LIB_CT = os.path.join(_HERE, "liboracle_corner_turn.so")
_SRC_DET = os.path.join(_HERE, "detect_oracle.cpp")
_LIB_DET = os.path.join(_HERE, "liboracle_detect.so")
_lib = None
_lib_ct = None
_lib_det = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-ffp-contract=off so ``fch1 + c*foff`` is never fused)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O3", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    if force or not os.path.exists(_LIB_CT) or os.path.getmtime(_LIB_CT) < os.path.getmtime(_SRC_CT):
        subprocess.run(["g++", "-O3", "-std=c++17", "-fPIC", "-shared", "-o", _LIB_CT, _SRC_CT], check=True)
    if force or not os.path.exists(_LIB_DET) or os.path.getmtime(_LIB_DET) < os.path.getmtime(_SRC_DET):
        subprocess.run(["g++", "-O3", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB_DET, _SRC_DET], check=True)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        plan = [ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double, dp]
        L.oracle_shift_table.argtypes = plan + [ctypes.c_int, ctypes.POINTER(ctypes.c_longlong)]
        L.oracle_shift_table.restype = ctypes.c_int
        L.oracle_max_shift.argtypes = plan + [ctypes.c_int]
        L.oracle_max_shift.restype = ctypes.c_longlong
        tail = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_longlong, ctypes.c_longlong]
        L.oracle_dedisperse_u8.argtypes = plan + [ip, ctypes.c_int] + tail + [ctypes.c_void_p]
        L.oracle_dedisperse_f32.argtypes = plan + [ip, ctypes.c_int] + tail + [ctypes.c_void_p, ctypes.c_void_p]
        L.oracle_dedisperse_f16.argtypes = plan + [ip, ctypes.c_int] + tail + [ctypes.c_void_p, ctypes.c_void_p]
        L.oracle_dedisperse_f32_seq.argtypes = plan + [ip, ctypes.c_int] + tail + [ctypes.c_void_p]
        for f in (L.oracle_dedisperse_u8, L.oracle_dedisperse_f32, L.oracle_dedisperse_f16,
                  L.oracle_dedisperse_f32_seq):
            f.restype = ctypes.c_int
        _lib = L
    return _lib


def _dm(dm_list):
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    return dm, dm.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def shift_table(nchans, fch1, foff, tsamp, dm_list) -> np.ndarray:
    """s(c,d) as int64 ``[nchans][ndm]``."""
    dm, dmp = _dm(dm_list)
    out = np.empty((nchans, dm.size), dtype=np.int64)
    rc = lib().oracle_shift_table(nchans, fch1, foff, tsamp, dmp, dm.size,
                                  out.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)))
    if rc:
        raise ValueError(f"oracle_shift_table rc={rc}")
    return out


def max_shift(nchans, fch1, foff, tsamp, dm_list) -> int:
    dm, dmp = _dm(dm_list)
    return int(lib().oracle_max_shift(nchans, fch1, foff, tsamp, dmp, dm.size))


def dedisperse(nchans, fch1, foff, tsamp, dm_list, data: np.ndarray, nsamp_out: int,
               rows=None, seq_f32: bool = False):
    """Run the oracle on ``data[nchans][nsamp_in]`` (uint8, float16 or float32).

    Returns int32 ``[nrows][nsamp_out]`` for uint8 input; ``(out_f64, abs_sum_f64)``
    for float input; float32 for ``seq_f32`` (diagnostic float accumulator).
    ``rows`` selects DM indices (default: all).
    """
    dm, dmp = _dm(dm_list)
    if rows is None:
        rows = np.arange(dm.size)
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    rp = rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
    assert data.ndim == 2 and data.shape[0] == nchans and data.flags.c_contiguous
    nsamp_in = data.shape[1]
    head = (nchans, fch1, foff, tsamp, dmp, rp, rows.size,
            data.ctypes.data, nsamp_in, nsamp_in, nsamp_out)
    L = lib()
    if data.dtype == np.uint8:
        out = np.empty((rows.size, nsamp_out), dtype=np.int32)
        rc = L.oracle_dedisperse_u8(*head, out.ctypes.data)
        res = out
    elif data.dtype == np.float32 and seq_f32:
        out = np.empty((rows.size, nsamp_out), dtype=np.float32)
        rc = L.oracle_dedisperse_f32_seq(*head, out.ctypes.data)
        res = out
    elif data.dtype in (np.float32, np.float16):
        out = np.empty((rows.size, nsamp_out), dtype=np.float64)
        asum = np.empty((rows.size, nsamp_out), dtype=np.float64)
        fn = L.oracle_dedisperse_f32 if data.dtype == np.float32 else L.oracle_dedisperse_f16
        rc = fn(*head, out.ctypes.data, asum.ctypes.data)
        res = (out, asum)
    else:
        raise TypeError(f"unsupported dtype {data.dtype}")
    if rc:
        raise ValueError(f"oracle dedisperse rc={rc}")
    return res


def unpack_time_major(raw: np.ndarray, nchans: int, nbits: int) -> np.ndarray:
    """``raw[nsamp][row_bytes]`` uint8 (time-major, ``nbits``-bit samples, first channel in the least
    significant bits) -> channel-major uint8 ``[nchans][nsamp]`` (oracle/corner_turn_oracle.cpp)."""
    global _lib_ct
    if _lib_ct is None:
        build()
        _lib_ct = ctypes.CDLL(_LIB_CT)
        _lib_ct.oracle_unpack_time_major.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_longlong, ctypes.c_int,
                                                      ctypes.c_int, ctypes.c_void_p, ctypes.c_longlong]
        _lib_ct.oracle_unpack_time_major.restype = ctypes.c_int
    assert raw.ndim == 2 and raw.dtype == np.uint8 and raw.flags.c_contiguous
    out = np.empty((nchans, raw.shape[0]), dtype=np.uint8)
    rc = _lib_ct.oracle_unpack_time_major(raw.ctypes.data, raw.shape[1], raw.shape[0], nchans, nbits, out.ctypes.data, raw.shape[0])
    if rc:
        raise ValueError(f"oracle_unpack_time_major rc={rc}")
    return out


CAND_DTYPE = np.dtype([("dm_index", np.int32), ("width", np.int32), ("t", np.int64), ("snr", np.float64)])


def detect(x: np.ndarray, nwidths: int, threshold: float, max_out: int = 1 << 20):
    """Detection oracle (oracle/detect_oracle.cpp) on ``x[nrows][n]`` (int32 or float32): returns
    (candidates as a CAND_DTYPE array in (row, width, t) order, total count)."""
    global _lib_det
    if _lib_det is None:
        build()
        _lib_det = ctypes.CDLL(_LIB_DET)
        for f in (_lib_det.oracle_detect_i32, _lib_det.oracle_detect_f32):
            f.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_double,
                          ctypes.c_void_p, ctypes.c_longlong]
            f.restype = ctypes.c_longlong
    assert x.ndim == 2 and x.flags.c_contiguous and x.dtype in (np.int32, np.float32)
    out = np.zeros(max_out, dtype=CAND_DTYPE)
    fn = _lib_det.oracle_detect_i32 if x.dtype == np.int32 else _lib_det.oracle_detect_f32
    n = fn(x.ctypes.data, x.shape[1], x.shape[0], x.shape[1], nwidths, float(threshold), out.ctypes.data, max_out)
    if n < 0:
        raise ValueError("oracle_detect: bad arguments")
    return out[:min(n, max_out)], int(n)
