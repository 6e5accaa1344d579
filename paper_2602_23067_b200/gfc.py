"""ctypes binding of the container layer of libb200gcm.so -- same names as include/gfc.h, marshalling only.

Host buffers are bytes / bytearray / numpy uint8 arrays / pinned torch CPU tensors.  The result's
data_buffer is pinned memory owned by the context: `FrameResult.view()` is a zero-copy numpy view that is
valid until the next call on the same context, `FrameResult.tobytes()` copies it out.
"""
from __future__ import annotations

import ctypes
from typing import Optional

import numpy as np

from . import gcm as _gcm
from .gcm import GCM_OK, GcmError

GFC_ERR_FORMAT, GFC_ERR_CAPACITY = -5, -6
GFC_FULL_ACCESS, GFC_HEADER_FALLBACK, GFC_PAYLOAD_SUPPRESSED = 0, 1, 2

EXPORTED_SYMBOLS = ["gfc_context_create", "gfc_context_destroy", "gfc_encrypt_frame", "gfc_decrypt_frame", "gfc_datasum",
                    "gfc_datasum_async", "gfc_datasum_noalloc"]
GFC_DATASUM_NOALLOC_MAX_BYTES = 1 << 32


class FitsOperationResult(ctypes.Structure):
    """struct FitsOperationResult of include/gfc.h (Table 1)"""
    _fields_ = [
        ("data_buffer", ctypes.c_void_p),
        ("buffer_size", ctypes.c_uint64),
        ("error_code", ctypes.c_int),
        ("warning_code", ctypes.c_int),
        ("header_ms", ctypes.c_float),
        ("data_ms", ctypes.c_float),
        ("error_message", ctypes.c_char * 128),
    ]


_L = _gcm._L
_vp, _u64, _ci = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int
_L.gfc_context_create.argtypes = [ctypes.POINTER(_vp), _u64, _u64]
_L.gfc_context_destroy.argtypes = [_vp]
_L.gfc_context_destroy.restype = None
_L.gfc_encrypt_frame.argtypes = [_vp, _vp, _u64, ctypes.c_char_p, ctypes.c_char_p, _ci, ctypes.c_char_p, ctypes.c_char_p,
                                 ctypes.POINTER(FitsOperationResult)]
_L.gfc_decrypt_frame.argtypes = [_vp, _vp, _u64, ctypes.c_char_p, ctypes.c_char_p, _ci, ctypes.POINTER(FitsOperationResult)]
_L.gfc_datasum.argtypes = [_vp, _u64, ctypes.POINTER(ctypes.c_uint32), _vp]
_L.gfc_datasum_async.argtypes = [_vp, _u64, _vp, _vp]
_L.gfc_datasum_noalloc.argtypes = [_vp, _u64, _vp, _vp]


class FrameError(GcmError):
    def __init__(self, code: int, where: str, message: str):
        RuntimeError.__init__(self, "%s failed with code %d: %s" % (where, code, message))
        self.code = code
        self.message = message


class FrameResult:
    def __init__(self, r: FitsOperationResult):
        self.data_buffer = r.data_buffer
        self.buffer_size = int(r.buffer_size)
        self.error_code = r.error_code
        self.warning_code = r.warning_code
        self.header_ms = float(r.header_ms)
        self.data_ms = float(r.data_ms)

    def view(self) -> np.ndarray:
        """Zero-copy view of the context-owned pinned buffer (valid until the next call on the context)."""
        buf = (ctypes.c_uint8 * self.buffer_size).from_address(self.data_buffer)
        return np.frombuffer(buf, dtype=np.uint8)

    def tobytes(self) -> bytes:
        return ctypes.string_at(self.data_buffer, self.buffer_size)


def _host_ptr(buf):
    """(address, nbytes, keep-alive) of a readable host buffer."""
    if isinstance(buf, (bytes, bytearray, memoryview)):
        a = np.frombuffer(buf, dtype=np.uint8)
        return a.ctypes.data, a.size, a
    if isinstance(buf, np.ndarray):
        a = np.ascontiguousarray(buf).view(np.uint8).reshape(-1)
        return a.ctypes.data, a.size, a
    if hasattr(buf, "data_ptr") and not getattr(buf, "is_cuda", False):
        return buf.data_ptr(), buf.numel() * buf.element_size(), buf
    raise TypeError("host buffer expected (bytes, numpy array or CPU tensor)")


def gfc_context_create(max_header_bytes: int, max_data_bytes: int) -> int:
    ctx = _vp()
    _gcm._check(_L.gfc_context_create(ctypes.byref(ctx), max_header_bytes, max_data_bytes), "gfc_context_create")
    return ctx.value


def gfc_context_destroy(ctx: Optional[int]) -> None:
    if ctx:
        _L.gfc_context_destroy(ctx)


def gfc_encrypt_frame(ctx: int, fits, key_h: bytes, key_d: bytes, nonce_h: Optional[bytes] = None,
                      nonce_d: Optional[bytes] = None) -> FrameResult:
    if len(key_h) != len(key_d) or len(key_h) not in (16, 32):
        raise ValueError("keys must both be 16 or both be 32 bytes")
    for n in (nonce_h, nonce_d):
        if n is not None and len(n) != 12:
            raise ValueError("nonces are 12 bytes")
    p, n, keep = _host_ptr(fits)
    r = FitsOperationResult()
    rc = _L.gfc_encrypt_frame(ctx, p, n, bytes(key_h), bytes(key_d), 8 * len(key_h), nonce_h, nonce_d, ctypes.byref(r))
    del keep
    if rc != GCM_OK:
        raise FrameError(rc, "gfc_encrypt_frame", r.error_message.decode("ascii", "replace"))
    return FrameResult(r)


def gfc_decrypt_frame(ctx: int, container, key_h: Optional[bytes], key_d: Optional[bytes]) -> FrameResult:
    """key_h / key_d = None: that key was not provisioned (Table 2)."""
    lens = {len(k) for k in (key_h, key_d) if k is not None}
    if len(lens) > 1 or (lens and lens.pop() not in (16, 32)):
        raise ValueError("keys must both be 16 or both be 32 bytes")
    bits = 8 * len(key_h if key_h is not None else key_d) if (key_h is not None or key_d is not None) else 0
    p, n, keep = _host_ptr(container)
    r = FitsOperationResult()
    rc = _L.gfc_decrypt_frame(ctx, p, n, None if key_h is None else bytes(key_h), None if key_d is None else bytes(key_d),
                              bits, ctypes.byref(r))
    del keep
    if rc != GCM_OK:
        raise FrameError(rc, "gfc_decrypt_frame", r.error_message.decode("ascii", "replace"))
    return FrameResult(r)


def gfc_datasum(d_data, stream=None) -> int:
    ptr, n = _gcm._dev(d_data)
    out = ctypes.c_uint32(0)
    _gcm._check(_L.gfc_datasum(ptr, n, ctypes.byref(out), _gcm._stream(stream)), "gfc_datasum")
    return int(out.value)


def gfc_datasum_async(d_data, d_acc, stream=None) -> None:
    """d_acc: device tensor holding one uint64 (8 bytes), zeroed by the caller; no synchronisation."""
    ptr, n = _gcm._dev(d_data)
    acc, _ = _gcm._dev(d_acc)
    _gcm._check(_L.gfc_datasum_async(ptr, n, acc, _gcm._stream(stream)), "gfc_datasum_async")


def gfc_datasum_noalloc(d_data, d_sum, stream=None) -> None:
    """DATASUM of a device buffer of at most 4 GiB without any device allocation inside the library.

    For programs in which the library may not call cudaMalloc: the GPU's memory is already owned by a caching
    allocator or a pre-reserved pool (a raw allocation would fail), or the call sits in a latency-critical loop
    beside other streams (cudaMalloc / cudaFree can stall the whole device).  The library's own scratch for this
    call is a fixed 128.25 KiB array inside its device image.

    d_sum: device tensor of 4 bytes (one uint32 / int32) owned by the caller; written asynchronously on
    `stream`, so synchronise (or order a later read on the same stream) before looking at it.  One call at a
    time per GPU: calls that could overlap on the device share the scratch and would corrupt each other.
    Raises GcmError(GCM_ERR_LEN) for more than GFC_DATASUM_NOALLOC_MAX_BYTES."""
    ptr, n = _gcm._dev(d_data)
    out, n_out = _gcm._dev(d_sum)
    if n_out != 4:
        raise ValueError("d_sum must be a device buffer of exactly 4 bytes")
    _gcm._check(_L.gfc_datasum_noalloc(ptr, n, out, _gcm._stream(stream)), "gfc_datasum_noalloc")
