"""Thin ctypes binding of ``libdedisp_b200.so`` (``include/dedisp.h``) — argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used to allocate device
tensors and to provide the current stream. There is no CPU fallback: if the library is missing it
is built with nvcc, and if that fails the import of this module raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np
import torch

from . import build as _build

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED, ETOOLARGE = 0, 1, 2, 3, 4, 5
DETECT_STATIC_MAX_NDM = 8192   # DEDISP_DETECT_STATIC_MAX_NDM
U8, F16, F32 = 0, 1, 2
KERNEL_AUTO, KERNEL_NAIVE, KERNEL_TILED, KERNEL_SUBBAND = 0, 1, 2, 3
PLAN_HOST_ONLY = 1
PLAN_TIME_MAJOR = 2
PLAN_NO_PACKED = 4

DTYPE_CODE = {"u8": U8, "f16": F16, "f32": F32}
_TORCH_IN = {U8: torch.uint8, F16: torch.float16, F32: torch.float32}
_TORCH_OUT = {U8: torch.int32, F16: torch.float32, F32: torch.float32}

# every symbol include/dedisp.h declares (tests check the library exports them all)
SYMBOLS = (
    "dedisp_shift_table_host", "dedisp_plan_create", "dedisp_plan_create_ex", "dedisp_execute",
    "dedisp_execute_strided", "dedisp_execute_batched", "dedisp_execute_host", "dedisp_execute_time_major", "dedisp_plan_destroy", "dedisp_plan_max_shift",
    "dedisp_plan_nchans", "dedisp_plan_ndm", "dedisp_plan_get_shifts", "dedisp_plan_set_kernel",
    "dedisp_plan_get_kernel", "dedisp_plan_set_pass_merge", "dedisp_plan_num_subbands", "dedisp_plan_get_subbands",
    "dedisp_plan_verify_records", "dedisp_plan_launches_per_execute", "dedisp_plan_last_host_slabs", "dedisp_plan_get_geometry", "dedisp_detect_workspace_bytes", "dedisp_detect", "dedisp_detect_static", "dedisp_error_string",
    "dedisp_last_cuda_error", "dedisp_stream_create", "dedisp_stream_push", "dedisp_stream_wait_event", "dedisp_stream_release_after", "dedisp_stream_sync",
    "dedisp_stream_destroy",
)

_lib: Optional[ctypes.CDLL] = None


class DedispError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        msg = lib().dedisp_error_string(code).decode()
        super().__init__(f"{what}: {msg} (code {code})" + (f" [{detail}]" if detail else ""))


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        c_int, c_ll, c_dbl, vp = ctypes.c_int, ctypes.c_longlong, ctypes.c_double, ctypes.c_void_p
        dp, ip = ctypes.POINTER(c_dbl), ctypes.POINTER(c_int)
        L.dedisp_shift_table_host.argtypes = [c_int, c_dbl, c_dbl, c_dbl, dp, c_int, ip, ctypes.POINTER(c_ll)]
        L.dedisp_plan_create.argtypes = [ctypes.POINTER(vp), c_int, c_dbl, c_dbl, c_dbl, dp, c_int, c_int]
        L.dedisp_plan_create_ex.argtypes = L.dedisp_plan_create.argtypes + [ctypes.c_uint]
        L.dedisp_execute.argtypes = [vp, vp, c_ll, vp, vp]
        L.dedisp_execute_strided.argtypes = [vp, vp, c_ll, c_ll, vp, c_ll, vp]
        L.dedisp_execute_batched.argtypes = [vp, c_int, vp, c_ll, c_ll, c_ll, vp, c_ll, c_ll, vp]
        L.dedisp_execute_host.argtypes = [vp, vp, c_ll, vp, vp]
        L.dedisp_execute_time_major.argtypes = [vp, vp, c_int, c_ll, c_ll, vp, vp]
        L.dedisp_plan_destroy.argtypes = [vp]
        L.dedisp_plan_max_shift.argtypes = [vp]
        L.dedisp_plan_max_shift.restype = c_ll
        for name in ("dedisp_plan_nchans", "dedisp_plan_ndm", "dedisp_plan_get_kernel", "dedisp_plan_set_pass_merge", "dedisp_plan_num_subbands",
                     "dedisp_plan_launches_per_execute", "dedisp_plan_last_host_slabs"):
            getattr(L, name).argtypes = [vp]
        L.dedisp_plan_get_shifts.argtypes = [vp, ip]
        L.dedisp_plan_set_kernel.argtypes = [vp, c_int]
        L.dedisp_plan_set_pass_merge.argtypes = [vp, c_int]
        L.dedisp_plan_get_subbands.argtypes = [vp, ip]
        L.dedisp_plan_get_geometry.argtypes = [vp, ip]
        L.dedisp_detect_workspace_bytes.argtypes = [c_int]
        L.dedisp_detect_workspace_bytes.restype = c_ll
        L.dedisp_detect.argtypes = [vp, c_int, c_int, c_ll, c_ll, c_int, c_dbl, vp, c_ll, vp, vp]
        L.dedisp_detect_static.argtypes = [vp, c_int, c_int, c_ll, c_ll, c_int, c_dbl, vp, c_ll, vp, vp]
        L.dedisp_plan_verify_records.argtypes = [vp]
        L.dedisp_plan_verify_records.restype = c_ll
        L.dedisp_error_string.argtypes = [c_int]
        L.dedisp_error_string.restype = ctypes.c_char_p
        L.dedisp_last_cuda_error.argtypes = [vp]
        L.dedisp_last_cuda_error.restype = ctypes.c_char_p
        L.dedisp_stream_create.argtypes = [ctypes.POINTER(vp), vp, c_int, c_ll, c_int]
        L.dedisp_stream_push.argtypes = [vp, vp, ctypes.POINTER(vp), ctypes.POINTER(vp)]
        L.dedisp_stream_wait_event.argtypes = [vp, vp]
        L.dedisp_stream_release_after.argtypes = [vp, vp]
        L.dedisp_stream_sync.argtypes = [vp]
        L.dedisp_stream_destroy.argtypes = [vp]
        _lib = L
    return _lib


def _dm(dm_list):
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    return dm, dm.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def shift_table_host(nchans, fch1, foff, tsamp, dm_list):
    """``dedisp_shift_table_host``: (int32 ``[nchans][ndm]``, maxshift). Pure host, no CUDA."""
    dm, dmp = _dm(dm_list)
    table = np.empty((nchans, dm.size), dtype=np.int32)
    mx = ctypes.c_longlong(0)
    rc = lib().dedisp_shift_table_host(nchans, fch1, foff, tsamp, dmp, dm.size,
                                       table.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), ctypes.byref(mx))
    if rc:
        raise DedispError(rc, "dedisp_shift_table_host")
    return table, int(mx.value)


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


class Plan:
    """``dedisp_plan``: shift table + kernel metadata for one (band, sampling, DM list, dtype)."""

    def __init__(self, nchans, fch1, foff, tsamp, dm_list, dtype, host_only: bool = False, time_major: bool = False, packed: bool = True):
        self._h = ctypes.c_void_p()
        self.dtype = DTYPE_CODE[dtype] if isinstance(dtype, str) else int(dtype)
        dm, dmp = _dm(dm_list)
        flags = (PLAN_HOST_ONLY if host_only else 0) | (PLAN_TIME_MAJOR if time_major else 0) | (0 if packed else PLAN_NO_PACKED)
        rc = lib().dedisp_plan_create_ex(ctypes.byref(self._h), int(nchans), float(fch1), float(foff), float(tsamp),
                                         dmp, dm.size, self.dtype, flags)
        if rc:
            self._h = ctypes.c_void_p()
            raise DedispError(rc, "dedisp_plan_create")
        self.nchans, self.ndm = int(nchans), int(dm.size)
        self.max_shift = int(lib().dedisp_plan_max_shift(self._h))

    @classmethod
    def from_config(cls, cfg, host_only: bool = False, time_major: bool = False, packed: bool = True) -> "Plan":
        return cls(cfg.nchans, cfg.fch1, cfg.foff, cfg.tsamp, cfg.dm_list(), cfg.dtype, host_only, time_major, packed)

    def _check(self, rc, what):
        if rc:
            raise DedispError(rc, what, lib().dedisp_last_cuda_error(self._h).decode())

    def shifts(self) -> np.ndarray:
        out = np.empty((self.nchans, self.ndm), dtype=np.int32)
        self._check(lib().dedisp_plan_get_shifts(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int))),
                    "dedisp_plan_get_shifts")
        return out

    def set_kernel(self, kernel: int) -> None:
        self._check(lib().dedisp_plan_set_kernel(self._h, int(kernel)), "dedisp_plan_set_kernel")

    def set_pass_merge(self, on: bool) -> None:
        """``dedisp_plan_set_pass_merge``: all SUBBAND passes in one launch (fp sums then not bit-reproducible)."""
        self._check(lib().dedisp_plan_set_pass_merge(self._h, int(bool(on))), "dedisp_plan_set_pass_merge")

    @property
    def kernel(self) -> int:
        return int(lib().dedisp_plan_get_kernel(self._h))

    @property
    def launches_per_execute(self) -> int:
        return int(lib().dedisp_plan_launches_per_execute(self._h))

    @property
    def last_host_slabs(self) -> int:
        return int(lib().dedisp_plan_last_host_slabs(self._h))

    def num_subbands(self) -> int:
        return int(lib().dedisp_plan_num_subbands(self._h))

    def subbands(self) -> np.ndarray:
        g = self.num_subbands()
        out = np.empty(g + 1, dtype=np.int32)
        self._check(lib().dedisp_plan_get_subbands(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int))),
                    "dedisp_plan_get_subbands")
        return out

    def geometry(self) -> dict:
        v = np.zeros(8, dtype=np.int32)
        self._check(lib().dedisp_plan_get_geometry(self._h, v.ctypes.data_as(ctypes.POINTER(ctypes.c_int))), "dedisp_plan_get_geometry")
        keys = ("cb", "cb_raw", "slot_bytes", "smem", "smem_raw", "nblk", "nranges", "npasses")
        return dict(zip(keys, (int(x) for x in v)))

    def verify_records(self) -> int:
        return int(lib().dedisp_plan_verify_records(self._h))

    def alloc_out(self, nsamp_out: int, nbeams: Optional[int] = None, device="cuda") -> torch.Tensor:
        shape = (self.ndm, nsamp_out) if nbeams is None else (nbeams, self.ndm, nsamp_out)
        return torch.empty(shape, dtype=_TORCH_OUT[self.dtype], device=device)

    def execute(self, d_in: torch.Tensor, nsamp_out: int, d_out: Optional[torch.Tensor] = None, stream=None):
        """``dedisp_execute`` / ``_strided`` / ``_batched`` on device tensors.

        ``d_in``: ``[nchans][>= nsamp_out + max_shift]`` or ``[nbeams][nchans][...]``, last dim
        contiguous; ``d_out`` likewise ``[ndm][>= nsamp_out]``. Asynchronous on ``stream``.
        """
        assert d_in.is_cuda and d_in.dtype == _TORCH_IN[self.dtype] and d_in.stride(-1) == 1
        batched = d_in.dim() == 3
        if d_out is None:
            d_out = self.alloc_out(nsamp_out, d_in.shape[0] if batched else None, d_in.device)
        assert d_out.is_cuda and d_out.dtype == _TORCH_OUT[self.dtype] and d_out.stride(-1) == 1
        assert d_in.shape[-2] == self.nchans and d_out.shape[-2] == self.ndm
        st = _stream_ptr(stream)
        if batched:
            assert d_out.dim() == 3 and d_out.shape[0] == d_in.shape[0]
            rc = lib().dedisp_execute_batched(self._h, d_in.shape[0], d_in.data_ptr(), d_in.stride(1), d_in.stride(0),
                                              nsamp_out, d_out.data_ptr(), d_out.stride(1), d_out.stride(0), st)
        else:
            rc = lib().dedisp_execute_strided(self._h, d_in.data_ptr(), d_in.stride(0) if self.nchans > 1 else d_in.shape[1],
                                              nsamp_out, d_out.data_ptr(),
                                              d_out.stride(0) if self.ndm > 1 else d_out.shape[1], st)
        self._check(rc, "dedisp_execute")
        return d_out

    def execute_time_major(self, d_raw: torch.Tensor, nbits: int, nsamp_out: int, d_out: Optional[torch.Tensor] = None, stream=None):
        """``dedisp_execute_time_major``: ``d_raw[nsamp_out + max_shift][row_bytes]`` uint8 on the device, time-major,
        ``nbits``-bit samples packed first-channel-in-the-low-bits; returns int32 ``[ndm][nsamp_out]``."""
        assert d_raw.is_cuda and d_raw.dtype == torch.uint8 and d_raw.dim() == 2 and d_raw.stride(1) == 1
        assert d_raw.shape[0] >= nsamp_out + self.max_shift
        if d_out is None:
            d_out = self.alloc_out(nsamp_out, None, d_raw.device)
        assert d_out.is_cuda and d_out.dtype == torch.int32 and d_out.is_contiguous()
        self._check(lib().dedisp_execute_time_major(self._h, d_raw.data_ptr(), int(nbits), d_raw.stride(0), nsamp_out,
                                                    d_out.data_ptr(), _stream_ptr(stream)), "dedisp_execute_time_major")
        return d_out

    def execute_host(self, h_in: torch.Tensor, nsamp_out: int, h_out: Optional[torch.Tensor] = None, stream=None):
        """``dedisp_execute_host``: host tensors in and out (pin them for full-speed copies); synchronous."""
        assert not h_in.is_cuda and h_in.is_contiguous() and h_in.dtype == _TORCH_IN[self.dtype]
        assert tuple(h_in.shape) == (self.nchans, nsamp_out + self.max_shift)
        if h_out is None:
            h_out = torch.empty((self.ndm, nsamp_out), dtype=_TORCH_OUT[self.dtype], pin_memory=True)
        assert not h_out.is_cuda and h_out.is_contiguous() and tuple(h_out.shape) == (self.ndm, nsamp_out)
        self._check(lib().dedisp_execute_host(self._h, h_in.data_ptr(), nsamp_out, h_out.data_ptr(),
                                              _stream_ptr(stream)), "dedisp_execute_host")
        return h_out

    def execute_raw(self, in_ptr: int, nsamp_out: int, out_ptr: int, stream=None) -> None:
        """``dedisp_execute`` on raw device pointers (dense rows)."""
        self._check(lib().dedisp_execute(self._h, in_ptr, nsamp_out, out_ptr, _stream_ptr(stream)), "dedisp_execute")

    def close(self) -> None:
        if getattr(self, "_h", None) and self._h.value:
            lib().dedisp_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class _DeviceBlob:
    """Exposes a raw device pointer through ``__cuda_array_interface__`` so torch can view it."""

    def __init__(self, ptr: int, shape, typestr: str):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2, "strides": None}


class Stream:
    """``dedisp_stream``: chunked multi-beam driver with H2D/compute overlap and maxshift carry."""

    def __init__(self, plan: Plan, nbeams: int, chunk_nsamp: int, nbuffers: int = 2):
        self._h = ctypes.c_void_p()
        self.plan, self.nbeams, self.chunk = plan, int(nbeams), int(chunk_nsamp)
        rc = lib().dedisp_stream_create(ctypes.byref(self._h), plan._h, self.nbeams, self.chunk, int(nbuffers))
        if rc:
            self._h = ctypes.c_void_p()
            raise DedispError(rc, "dedisp_stream_create", lib().dedisp_last_cuda_error(plan._h).decode())

    def push(self, h_chunk: torch.Tensor):
        """Enqueue ``h_chunk[beam][chan][chunk]`` (host, ideally pinned). Returns (out_ptr, event_ptr)."""
        assert not h_chunk.is_cuda and h_chunk.is_contiguous() and h_chunk.dtype == _TORCH_IN[self.plan.dtype]
        assert tuple(h_chunk.shape) == (self.nbeams, self.plan.nchans, self.chunk)
        out, ev = ctypes.c_void_p(), ctypes.c_void_p()
        self.plan._check(lib().dedisp_stream_push(self._h, h_chunk.data_ptr(), ctypes.byref(out), ctypes.byref(ev)),
                         "dedisp_stream_push")
        return out.value, ev.value

    def out_view(self, out_ptr: int) -> torch.Tensor:
        """Zero-copy torch view ``[beam][ndm][chunk]`` of an output block owned by the stream object."""
        typestr = "<i4" if self.plan.dtype == U8 else "<f4"
        return torch.as_tensor(_DeviceBlob(out_ptr, (self.nbeams, self.plan.ndm, self.chunk), typestr), device="cuda")

    def wait_event(self, event_ptr: int, stream=None) -> None:
        """``dedisp_stream_wait_event``: ``stream`` (default: torch's current) waits for a block's done event."""
        self.plan._check(lib().dedisp_stream_wait_event(event_ptr, _stream_ptr(stream)), "dedisp_stream_wait_event")

    def release_after(self, event: "torch.cuda.Event") -> None:
        """Later pushes compute after `event` (recorded by the consumer after its last read of a block)."""
        self.plan._check(lib().dedisp_stream_release_after(self._h, ctypes.c_void_p(event.cuda_event)),
                         "dedisp_stream_release_after")

    def sync(self) -> None:
        self.plan._check(lib().dedisp_stream_sync(self._h), "dedisp_stream_sync")

    def close(self) -> None:
        if getattr(self, "_h", None) and self._h.value:
            lib().dedisp_stream_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


CAND_DTYPE = np.dtype([("dm_index", np.int32), ("width", np.int32), ("t", np.int64), ("snr", np.float64)])


def detect(block: torch.Tensor, nwidths: int, threshold: float, max_cands: int = 1 << 20, stream=None):
    """``dedisp_detect`` on a de-dispersed block ``[ndm][nsamp]`` (int32 or float32, device). Returns
    (candidates as a CAND_DTYPE numpy array, total count). Marshalling only: buffers, call, copy back."""
    assert block.is_cuda and block.dim() == 2 and block.stride(1) == 1 and block.dtype in (torch.int32, torch.float32)
    ndm, nsamp = block.shape
    work = torch.empty(int(lib().dedisp_detect_workspace_bytes(ndm)) // 8 + 1, dtype=torch.int64, device=block.device)
    cands = torch.empty(max(1, max_cands) * CAND_DTYPE.itemsize, dtype=torch.uint8, device=block.device)
    rc = lib().dedisp_detect(block.data_ptr(), int(block.dtype == torch.float32), ndm, nsamp, block.stride(0), int(nwidths),
                             float(threshold), cands.data_ptr(), int(max_cands), work.data_ptr(), _stream_ptr(stream))
    if rc:
        raise DedispError(rc, "dedisp_detect")
    torch.cuda.synchronize(block.device)
    total = int(work[0].item())
    out = np.frombuffer(cands[:min(total, max_cands) * CAND_DTYPE.itemsize].cpu().numpy().tobytes(), dtype=CAND_DTYPE)
    return out, total


def detect_static(block: torch.Tensor, nwidths: int, threshold: float, max_cands: int = 1 << 20, stream=None,
                  cands: Optional[torch.Tensor] = None, count: Optional[torch.Tensor] = None):
    """``dedisp_detect_static``: ``detect`` without a workspace - the library call allocates nothing, its scratch is a
    fixed ``static __device__`` array (at most DETECT_STATIC_MAX_NDM rows; calls that overlap on the GPU race).
    The outputs are the caller's: pass ``cands`` (uint8, >= max_cands records) and ``count`` (int64[1]) to reuse
    buffers, else they are made here. Returns (candidates as a CAND_DTYPE numpy array, total count)."""
    assert block.is_cuda and block.dim() == 2 and block.stride(1) == 1 and block.dtype in (torch.int32, torch.float32)
    ndm, nsamp = block.shape
    if cands is None:
        cands = torch.empty(max(1, max_cands) * CAND_DTYPE.itemsize, dtype=torch.uint8, device=block.device)
    if count is None:
        count = torch.empty(1, dtype=torch.int64, device=block.device)
    assert cands.is_cuda and cands.numel() * cands.element_size() >= max_cands * CAND_DTYPE.itemsize
    assert count.is_cuda and count.dtype == torch.int64 and count.numel() >= 1
    rc = lib().dedisp_detect_static(block.data_ptr(), int(block.dtype == torch.float32), ndm, nsamp, block.stride(0), int(nwidths),
                                    float(threshold), cands.data_ptr(), int(max_cands), count.data_ptr(), _stream_ptr(stream))
    if rc:
        raise DedispError(rc, "dedisp_detect_static")
    torch.cuda.synchronize(block.device)
    total = int(count[0].item())
    flat = cands.view(torch.uint8).reshape(-1)
    out = np.frombuffer(flat[:min(total, max_cands) * CAND_DTYPE.itemsize].cpu().numpy().tobytes(), dtype=CAND_DTYPE)
    return out, total
