"""ctypes binding of libb200gcm.so -- same names as include/gcm.h, marshalling only.

Device buffers are torch uint8 CUDA tensors (PyTorch is used for device memory and streams only);
anything exposing data_ptr()/numel() works, and plain ints are taken as raw device addresses.
Every step of the path (key schedule, H powers, CTR, GHASH, tag, compare, wipe) runs in the
library's CUDA kernels.  If the library is missing this module raises: there is no fallback.
"""
from __future__ import annotations

import ctypes
import os
from typing import Iterable, List, Optional, Sequence, Tuple

GCM_OK, GCM_ERR_AUTH, GCM_ERR_ARG, GCM_ERR_LEN, GCM_ERR_CUDA, GCM_ERR_NOMEM, GCM_ERR_BUSY = 0, 1, -1, -2, -3, -4, -5
GCM_PHASE_SLOTS = 8
GCM_GHASH_TABLE = 0
GCM_GHASH_TENSOR = 1
GCM_GHASH_AUTO = 2
# sizes from which GCM_GHASH_AUTO takes the tensor-core kernels (csrc/gcm_common.cuh: T2_AUTO_BYTES_*, GT_AUTO_BYTES)
TC2_AUTO_BYTES = {128: 128 << 20, 256: 384 << 20}
GHASH_TC_AUTO_BYTES = 32 << 20

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libb200gcm.so")

EXPORTED_SYMBOLS = [
    "gcm_version", "gcm_set_device", "gcm_last_cuda_error", "gcm_last_cuda_error_string",
    "gcm_init", "gcm_destroy", "gcm_set_geometry", "gcm_get_geometry", "gcm_set_ghash_engine", "gcm_get_ghash_engine", "gcm_get_hash_subkey",
    "gcm_encrypt", "gcm_decrypt_verify", "gcm_encrypt_async", "gcm_decrypt_verify_async",
    "gcm_encrypt_host", "gcm_decrypt_verify_host", "gcm_decrypt_verify_host_strict", "gcm_set_phase_stamps",
    "gcm_ghash_async", "gcm_encrypt_batch", "gcm_decrypt_verify_batch", "gcm_batch_release",
    "gcm_encrypt_batch_device", "gcm_decrypt_verify_batch_device", "gcm_debug_row_layout", "gcm_debug_plan_chunks", "gcm_debug_tc2_clock",
    "gcm_measure_pipe_rates",
]
RATE_NAMES = ["lds32", "lds128", "lop3", "prmt", "imad", "imad_wide", "lop3_imad", "mma_mxf4_blocks"]


class GcmError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        detail = ""
        if code == GCM_ERR_CUDA:
            detail = ": " + gcm_last_cuda_error_string()
        super().__init__("%s failed with code %d%s" % (where, code, detail))


class GcmRowLayout(ctypes.Structure):
    """struct gcm_row_layout of include/gcm.h"""
    _fields_ = [("vblocks", ctypes.c_uint64), ("base", ctypes.c_uint64), ("pad", ctypes.c_uint32),
                ("n_aad_blocks", ctypes.c_uint32), ("rows", ctypes.c_uint32), ("fast_lo", ctypes.c_uint32),
                ("fast_hi", ctypes.c_uint32), ("ctr_delta", ctypes.c_uint32), ("len_block", ctypes.c_uint32),
                ("reserved", ctypes.c_uint32)]


class GcmMsg(ctypes.Structure):
    """struct gcm_msg of include/gcm.h"""
    _fields_ = [
        ("key", ctypes.c_void_p),
        ("key_bits", ctypes.c_int),
        ("iv", ctypes.c_uint8 * 12),
        ("d_aad", ctypes.c_void_p),
        ("aad_len", ctypes.c_uint64),
        ("d_in", ctypes.c_void_p),
        ("len", ctypes.c_uint64),
        ("d_out", ctypes.c_void_p),
        ("tag", ctypes.c_uint8 * 16),
        ("status", ctypes.c_int),
    ]


def library_path() -> str:
    return _LIB_PATH


def _load() -> ctypes.CDLL:
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            "libb200gcm.so is not built (%s). Run `python -m paper_2602_23067_b200.build` "
            "(needs nvcc); there is no CPU fallback." % _LIB_PATH)
    L = ctypes.CDLL(_LIB_PATH)
    vp, u64, ci = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int
    L.gcm_version.restype = ctypes.c_char_p
    L.gcm_version.argtypes = []
    L.gcm_set_device.argtypes = [ci]
    L.gcm_last_cuda_error.argtypes = []
    L.gcm_last_cuda_error_string.restype = ctypes.c_char_p
    L.gcm_last_cuda_error_string.argtypes = []
    L.gcm_init.argtypes = [ctypes.POINTER(vp), ctypes.c_char_p, ci]
    L.gcm_destroy.argtypes = [vp]
    L.gcm_destroy.restype = None
    L.gcm_set_geometry.argtypes = [vp, ci, ci]
    L.gcm_get_geometry.argtypes = [vp, ctypes.POINTER(ci), ctypes.POINTER(ci)]
    L.gcm_set_ghash_engine.argtypes = [vp, ci]
    L.gcm_get_ghash_engine.argtypes = [vp, ctypes.POINTER(ci)]
    L.gcm_get_hash_subkey.argtypes = [vp, ctypes.c_char_p]
    L.gcm_encrypt.argtypes = [vp, ctypes.c_char_p, vp, u64, vp, u64, vp, ctypes.c_char_p, vp]
    L.gcm_decrypt_verify.argtypes = [vp, ctypes.c_char_p, vp, u64, vp, u64, vp, ctypes.c_char_p, vp]
    L.gcm_encrypt_async.argtypes = [vp, ctypes.c_char_p, vp, u64, vp, u64, vp, vp, vp]
    L.gcm_decrypt_verify_async.argtypes = [vp, ctypes.c_char_p, vp, u64, vp, u64, vp, vp, vp, vp]
    L.gcm_ghash_async.argtypes = [vp, vp, u64, vp, u64, vp, vp]
    L.gcm_encrypt_host.argtypes = [vp, ctypes.c_char_p, vp, u64, vp, u64, vp, ctypes.c_char_p, vp]
    L.gcm_decrypt_verify_host.argtypes = [vp, ctypes.c_char_p, vp, u64, vp, u64, vp, ctypes.c_char_p, vp]
    L.gcm_decrypt_verify_host_strict.argtypes = [vp, ctypes.c_char_p, vp, u64, vp, u64, vp, ctypes.c_char_p, vp]
    L.gcm_set_phase_stamps.argtypes = [vp, vp]
    L.gcm_encrypt_batch.argtypes = [ctypes.POINTER(GcmMsg), ctypes.c_uint32, vp]
    L.gcm_decrypt_verify_batch.argtypes = [ctypes.POINTER(GcmMsg), ctypes.c_uint32, vp]
    L.gcm_encrypt_batch_device.argtypes = [vp, ctypes.c_uint32, vp]
    L.gcm_decrypt_verify_batch_device.argtypes = [vp, ctypes.c_uint32, vp]
    L.gcm_debug_row_layout.argtypes = [u64, u64, ctypes.c_uint32, ci, ci, ctypes.POINTER(GcmRowLayout)]
    L.gcm_debug_plan_chunks.argtypes = [u64, ctypes.POINTER(u64), ctypes.c_uint32]
    L.gcm_debug_tc2_clock.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.gcm_batch_release.argtypes = []
    L.gcm_batch_release.restype = None
    L.gcm_measure_pipe_rates.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.c_int]
    L.gcm_measure_pipe_rates.restype = ctypes.c_int
    return L


_L = _load()


# ---- marshalling ---------------------------------------------------------------------------------
def _dev(buf) -> Tuple[Optional[int], int]:
    """(device address or None, byte length) of a device buffer argument."""
    if buf is None:
        return None, 0
    if isinstance(buf, int):
        raise TypeError("raw device addresses need an explicit length; pass (ptr, nbytes)")
    if isinstance(buf, tuple):
        return (int(buf[0]) or None), int(buf[1])
    if not getattr(buf, "is_cuda", False):
        raise TypeError("device buffer expected (torch CUDA tensor)")
    if not buf.is_contiguous():
        raise ValueError("device buffer must be contiguous")
    n = buf.numel() * buf.element_size()
    return (buf.data_ptr() if n else None), n


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


def _iv(iv) -> bytes:
    """The C side reads exactly 12 bytes (include/gcm.h: 96-bit IV only, reading S5): refuse anything else here,
    a short IV would be read past its end and a longer one silently truncated (nonce collisions)."""
    iv = bytes(iv)
    if len(iv) != 12:
        raise ValueError("iv must be exactly 12 bytes (96 bits), got %d" % len(iv))
    return iv


def _tag(tag) -> bytes:
    tag = bytes(tag)
    if len(tag) != 16:
        raise ValueError("tag must be exactly 16 bytes, got %d" % len(tag))
    return tag


def _check(rc: int, where: str, ok: Sequence[int] = (GCM_OK,)) -> int:
    if rc not in ok:
        raise GcmError(rc, where)
    return rc


# ---- the C ABI, one function per entry point -----------------------------------------------------
def gcm_version() -> str:
    return _L.gcm_version().decode()


def gcm_set_device(ordinal: int) -> None:
    _check(_L.gcm_set_device(int(ordinal)), "gcm_set_device")


def gcm_last_cuda_error() -> int:
    return _L.gcm_last_cuda_error()


def gcm_last_cuda_error_string() -> str:
    return _L.gcm_last_cuda_error_string().decode()


def gcm_init(key: bytes, key_bits: Optional[int] = None) -> int:
    key = bytes(key)
    bits = 8 * len(key) if key_bits is None else int(key_bits)
    if bits not in (128, 256) or 8 * len(key) != bits:
        raise ValueError("key must be 16 or 32 bytes and match key_bits (got %d bytes, key_bits=%d)" % (len(key), bits))
    h = ctypes.c_void_p()
    _check(_L.gcm_init(ctypes.byref(h), key, bits), "gcm_init")
    return h.value


def gcm_destroy(ctx: Optional[int]) -> None:
    if ctx:
        _L.gcm_destroy(ctx)


def gcm_set_geometry(ctx: int, grid: int = 0, threads: int = 0) -> None:
    _check(_L.gcm_set_geometry(ctx, int(grid), int(threads)), "gcm_set_geometry")


def gcm_get_geometry(ctx: int) -> Tuple[int, int]:
    g, t = ctypes.c_int(), ctypes.c_int()
    _check(_L.gcm_get_geometry(ctx, ctypes.byref(g), ctypes.byref(t)), "gcm_get_geometry")
    return g.value, t.value


def gcm_set_ghash_engine(ctx: int, engine: int) -> None:
    _check(_L.gcm_set_ghash_engine(ctx, int(engine)), "gcm_set_ghash_engine")


def gcm_get_ghash_engine(ctx: int) -> int:
    e = ctypes.c_int()
    _check(_L.gcm_get_ghash_engine(ctx, ctypes.byref(e)), "gcm_get_ghash_engine")
    return e.value


def gcm_get_hash_subkey(ctx: int) -> bytes:
    buf = ctypes.create_string_buffer(16)
    _check(_L.gcm_get_hash_subkey(ctx, buf), "gcm_get_hash_subkey")
    return buf.raw


def gcm_encrypt(ctx: int, iv: bytes, aad, pt, ct, stream=None) -> bytes:
    """Encrypts device buffer `pt` into device buffer `ct` (same size; may be the same tensor) and
    returns the 16-byte tag."""
    iv = _iv(iv)
    a_ptr, a_len = _dev(aad)
    p_ptr, p_len = _dev(pt)
    c_ptr, c_len = _dev(ct)
    if c_len != p_len:
        raise ValueError("ct and pt sizes differ")
    tag = ctypes.create_string_buffer(16)
    _check(_L.gcm_encrypt(ctx, iv, a_ptr, a_len, p_ptr, p_len, c_ptr, tag, _stream(stream)), "gcm_encrypt")
    return tag.raw


def gcm_decrypt_verify(ctx: int, iv: bytes, aad, ct, pt, tag: bytes, stream=None) -> int:
    """Returns GCM_OK (plaintext in `pt`) or GCM_ERR_AUTH (`pt` zero-filled)."""
    iv, tag = _iv(iv), _tag(tag)
    a_ptr, a_len = _dev(aad)
    c_ptr, c_len = _dev(ct)
    p_ptr, p_len = _dev(pt)
    if c_len != p_len:
        raise ValueError("ct and pt sizes differ")
    return _check(_L.gcm_decrypt_verify(ctx, iv, a_ptr, a_len, c_ptr, c_len, p_ptr, tag, _stream(stream)),
                  "gcm_decrypt_verify", ok=(GCM_OK, GCM_ERR_AUTH))


def gcm_encrypt_async(ctx: int, iv: bytes, aad, pt, ct, d_tag, stream=None) -> None:
    iv = _iv(iv)
    a_ptr, a_len = _dev(aad)
    p_ptr, p_len = _dev(pt)
    c_ptr, _ = _dev(ct)
    t_ptr, t_len = _dev(d_tag)
    if t_len < 16:
        raise ValueError("d_tag must hold 16 bytes")
    _check(_L.gcm_encrypt_async(ctx, iv, a_ptr, a_len, p_ptr, p_len, c_ptr, t_ptr, _stream(stream)),
           "gcm_encrypt_async")


def gcm_decrypt_verify_async(ctx: int, iv: bytes, aad, ct, pt, d_tag, d_status, stream=None) -> None:
    iv = _iv(iv)
    a_ptr, a_len = _dev(aad)
    c_ptr, c_len = _dev(ct)
    p_ptr, _ = _dev(pt)
    t_ptr, t_len = _dev(d_tag)
    s_ptr, s_len = _dev(d_status)
    if t_len < 16 or s_len < 4:
        raise ValueError("d_tag must hold 16 bytes and d_status 4")
    _check(_L.gcm_decrypt_verify_async(ctx, iv, a_ptr, a_len, c_ptr, c_len, p_ptr, t_ptr, s_ptr,
                                       _stream(stream)), "gcm_decrypt_verify_async")


def _host(buf, writable: bool = False) -> Tuple[Optional[int], int, object]:
    """(address or None, byte length, keep-alive) of a HOST buffer: numpy array, CPU torch tensor
    (pinned or not), bytes / bytearray / memoryview."""
    if buf is None:
        return None, 0, None
    if hasattr(buf, "data_ptr"):
        if getattr(buf, "is_cuda", False):
            raise TypeError("host buffer expected, got a CUDA tensor")
        if not buf.is_contiguous():
            raise ValueError("host buffer must be contiguous")
        n = buf.numel() * buf.element_size()
        return (buf.data_ptr() if n else None), n, buf
    import numpy as np
    if isinstance(buf, np.ndarray):
        if not buf.flags["C_CONTIGUOUS"] or (writable and not buf.flags["WRITEABLE"]):
            raise ValueError("host array must be contiguous (and writable for outputs)")
        return (buf.ctypes.data if buf.nbytes else None), buf.nbytes, buf
    if writable:
        raise TypeError("writable host buffer expected (numpy array or CPU tensor)")
    arr = np.frombuffer(bytes(buf), dtype=np.uint8)
    return (arr.ctypes.data if arr.size else None), arr.size, arr


def gcm_encrypt_host(ctx: int, iv: bytes, h_aad, h_pt, h_ct, stream=None) -> bytes:
    """HOST buffers in and out (chunked H2D -> kernel -> D2H pipeline inside the library)."""
    iv = _iv(iv)
    a_ptr, a_len, ka = _host(h_aad)
    p_ptr, p_len, kp = _host(h_pt)
    c_ptr, c_len, kc = _host(h_ct, writable=True)
    if c_len != p_len:
        raise ValueError("ct and pt sizes differ")
    tag = ctypes.create_string_buffer(16)
    _check(_L.gcm_encrypt_host(ctx, iv, a_ptr, a_len, p_ptr, p_len, c_ptr, tag, _stream(stream)),
           "gcm_encrypt_host")
    del ka, kp, kc
    return tag.raw


def gcm_decrypt_verify_host(ctx: int, iv: bytes, h_aad, h_ct, h_pt, tag: bytes, stream=None) -> int:
    iv, tag = _iv(iv), _tag(tag)
    a_ptr, a_len, ka = _host(h_aad)
    c_ptr, c_len, kc = _host(h_ct)
    p_ptr, p_len, kp = _host(h_pt, writable=True)
    if c_len != p_len:
        raise ValueError("ct and pt sizes differ")
    rc = _check(_L.gcm_decrypt_verify_host(ctx, iv, a_ptr, a_len, c_ptr, c_len, p_ptr, tag, _stream(stream)),
                "gcm_decrypt_verify_host", ok=(GCM_OK, GCM_ERR_AUTH))
    del ka, kp, kc
    return rc


def gcm_decrypt_verify_host_strict(ctx: int, iv: bytes, h_aad, h_ct, h_pt, tag: bytes, stream=None) -> int:
    """Verify-then-release: h_pt is written only after the tag has been verified (two passes over h_ct)."""
    iv, tag = _iv(iv), _tag(tag)
    a_ptr, a_len, ka = _host(h_aad)
    c_ptr, c_len, kc = _host(h_ct)
    p_ptr, p_len, kp = _host(h_pt, writable=True)
    if c_len != p_len:
        raise ValueError("ct and pt sizes differ")
    rc = _check(_L.gcm_decrypt_verify_host_strict(ctx, iv, a_ptr, a_len, c_ptr, c_len, p_ptr, tag, _stream(stream)),
                "gcm_decrypt_verify_host_strict", ok=(GCM_OK, GCM_ERR_AUTH))
    del ka, kp, kc
    return rc


def gcm_set_phase_stamps(ctx: int, d_stamps) -> None:
    """Diagnostics: d_stamps = device buffer of GCM_PHASE_SLOTS x grid uint64 (or None to switch it off)."""
    ptr, n = _dev(d_stamps)
    _check(_L.gcm_set_phase_stamps(ctx, ptr), "gcm_set_phase_stamps")


def gcm_ghash_async(ctx: int, aad, c, d_out, stream=None) -> None:
    a_ptr, a_len = _dev(aad)
    c_ptr, c_len = _dev(c)
    o_ptr, o_len = _dev(d_out)
    if o_len < 16:
        raise ValueError("d_out must hold 16 bytes")
    _check(_L.gcm_ghash_async(ctx, a_ptr, a_len, c_ptr, c_len, o_ptr, _stream(stream)), "gcm_ghash_async")


def _pack_msgs(msgs: Iterable[dict], decrypt: bool):
    msgs = list(msgs)
    arr = (GcmMsg * max(1, len(msgs)))()
    keep = []
    for i, m in enumerate(msgs):
        key = ctypes.create_string_buffer(bytes(m["key"]), len(m["key"]))
        keep.append(key)
        arr[i].key = ctypes.cast(key, ctypes.c_void_p)
        arr[i].key_bits = 8 * len(m["key"])
        arr[i].iv[:] = list(_iv(m["iv"]))
        a_ptr, a_len = _dev(m.get("aad"))
        i_ptr, i_len = _dev(m["input"])
        o_ptr, o_len = _dev(m["output"])
        if o_len != i_len:
            raise ValueError("message %d: input and output sizes differ" % i)
        arr[i].d_aad, arr[i].aad_len = a_ptr, a_len
        arr[i].d_in, arr[i].len = i_ptr, i_len
        arr[i].d_out = o_ptr
        if decrypt:
            arr[i].tag[:] = list(_tag(m["tag"]))
    return arr, len(msgs), keep


class MsgBatch:
    """The gcm_msg array of include/gcm.h, built once from a list of dicts (gcm_pack_msgs) so that a batch which is
    submitted many times pays the Python-side marshalling once.  Keeps the key buffers (and nothing else) alive: the
    device buffers the descriptors point to stay the caller's."""

    def __init__(self, msgs: Iterable[dict], decrypt: bool):
        self.decrypt = bool(decrypt)
        self.arr, self.n, self._keep = _pack_msgs(msgs, decrypt)

    def __len__(self) -> int:
        return self.n


def gcm_pack_msgs(msgs: Iterable[dict], decrypt: bool = False) -> MsgBatch:
    """dicts with key, iv, aad (device or None), input, output (device) and, for decrypt, tag -> MsgBatch."""
    return MsgBatch(msgs, decrypt)


def gcm_encrypt_batch(msgs, stream=None) -> List[bytes]:
    """msgs: dicts with key, iv, aad (device or None), input, output (device), or a MsgBatch.  Returns the tags."""
    b = msgs if isinstance(msgs, MsgBatch) else MsgBatch(msgs, decrypt=False)
    if b.decrypt:
        raise ValueError("a MsgBatch packed for decrypt was passed to gcm_encrypt_batch")
    _check(_L.gcm_encrypt_batch(b.arr, b.n, _stream(stream)), "gcm_encrypt_batch")
    return [bytes(b.arr[i].tag) for i in range(b.n)]


def gcm_decrypt_verify_batch(msgs, stream=None) -> List[int]:
    """msgs as above plus `tag` (or a MsgBatch packed with decrypt=True).  Returns the per-message status list
    (GCM_OK / GCM_ERR_AUTH)."""
    b = msgs if isinstance(msgs, MsgBatch) else MsgBatch(msgs, decrypt=True)
    if not b.decrypt:
        raise ValueError("a MsgBatch packed for encrypt was passed to gcm_decrypt_verify_batch")
    rc = _L.gcm_decrypt_verify_batch(b.arr, b.n, _stream(stream))
    if rc < 0:
        raise GcmError(rc, "gcm_decrypt_verify_batch")
    return [b.arr[i].status for i in range(b.n)]


GCM_DMSG_BYTES = 112


def gcm_dmsg_dtype():
    """numpy structured dtype of struct gcm_dmsg (include/gcm.h), 112 bytes."""
    import numpy as np
    return np.dtype([("key", np.uint8, 32), ("tag", np.uint8, 16), ("status", np.int32), ("key_bits", np.uint32),
                     ("iv", np.uint8, 12), ("reserved", np.uint32), ("d_aad", np.uint64), ("d_in", np.uint64),
                     ("d_out", np.uint64), ("aad_len", np.uint64), ("len", np.uint64)])


def gcm_pack_dmsgs(msgs: Iterable[dict]):
    """Host array of gcm_dmsg records from dicts with key, iv, aad (device or None), input, output (device) and, for
    decryption, tag.  Marshalling only; copy it to the device (torch.from_numpy(a.view(numpy.uint8)).cuda()) and hand
    that tensor to gcm_encrypt_batch_device / gcm_decrypt_verify_batch_device."""
    import numpy as np
    msgs = list(msgs)
    a = np.zeros(len(msgs), dtype=gcm_dmsg_dtype())
    assert a.dtype.itemsize == GCM_DMSG_BYTES
    for i, m in enumerate(msgs):
        key = bytes(m["key"])
        a["key"][i, :len(key)] = np.frombuffer(key, np.uint8)[:32]
        a["key_bits"][i] = 8 * len(key)
        a["iv"][i] = np.frombuffer(_iv(m["iv"]), np.uint8)
        a_ptr, a_len = _dev(m.get("aad"))
        i_ptr, i_len = _dev(m["input"])
        o_ptr, o_len = _dev(m["output"])
        if o_len != i_len:
            raise ValueError("message %d: input and output sizes differ" % i)
        a["d_aad"][i], a["aad_len"][i] = a_ptr or 0, a_len
        a["d_in"][i], a["len"][i] = i_ptr or 0, i_len
        a["d_out"][i] = o_ptr or 0
        if "tag" in m and m["tag"] is not None:
            a["tag"][i] = np.frombuffer(_tag(m["tag"]), np.uint8)
    return a


def _dmsgs(d_msgs, n):
    ptr, nbytes = _dev(d_msgs)
    if n is None:
        n = nbytes // GCM_DMSG_BYTES
    if nbytes < n * GCM_DMSG_BYTES:
        raise ValueError("d_msgs holds fewer than n descriptors")
    return ptr, int(n)


def gcm_encrypt_batch_device(d_msgs, n: Optional[int] = None, stream=None) -> None:
    """Asynchronous; tags and statuses land in the device-resident descriptors (gcm_dmsg)."""
    ptr, n = _dmsgs(d_msgs, n)
    _check(_L.gcm_encrypt_batch_device(ptr, n, _stream(stream)), "gcm_encrypt_batch_device")


def gcm_decrypt_verify_batch_device(d_msgs, n: Optional[int] = None, stream=None) -> None:
    ptr, n = _dmsgs(d_msgs, n)
    _check(_L.gcm_decrypt_verify_batch_device(ptr, n, _stream(stream)), "gcm_decrypt_verify_batch_device")


def gcm_debug_row_layout(length: int, aad_len: int, ctr_base: int = 0, last: bool = True, aligned: bool = True) -> dict:
    out = GcmRowLayout()
    _check(_L.gcm_debug_row_layout(length, aad_len, ctr_base, 1 if last else 0, 1 if aligned else 0, ctypes.byref(out)),
           "gcm_debug_row_layout")
    return {k: getattr(out, k) for k, _ in GcmRowLayout._fields_ if k != "reserved"}


def gcm_debug_tc2_clock(ctx: int) -> Tuple[float, float]:
    """(SM MHz, kernel ms) of gcm_tc2_kernel in the context's most recent long-message call, measured by the kernel."""
    mhz, ms = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(_L.gcm_debug_tc2_clock(ctx, ctypes.byref(mhz), ctypes.byref(ms)), "gcm_debug_tc2_clock")
    return float(mhz.value), float(ms.value)


def gcm_debug_plan_chunks(length: int) -> List[int]:
    cap = 1200
    plan = (ctypes.c_uint64 * cap)()
    n = _L.gcm_debug_plan_chunks(length, plan, cap)
    if n < 0:
        raise GcmError(n, "gcm_debug_plan_chunks")
    return [int(plan[i]) for i in range(n)]


def gcm_batch_release() -> None:
    _L.gcm_batch_release()


def gcm_measure_pipe_rates() -> dict:
    """Thread-operations per SM-cycle of the instruction classes in RATE_NAMES, measured on the device."""
    out = (ctypes.c_double * len(RATE_NAMES))()
    _check(_L.gcm_measure_pipe_rates(out, len(RATE_NAMES)), "gcm_measure_pipe_rates")
    return {k: float(out[i]) for i, k in enumerate(RATE_NAMES)}


class Context:
    """Owns one gcm_ctx.  Convenience wrapper over the functions above."""

    def __init__(self, key: bytes):
        self.handle = gcm_init(key)
        self.key_bits = 8 * len(key)

    def close(self) -> None:
        if self.handle:
            gcm_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_geometry(self, grid: int = 0, threads: int = 0) -> None:
        gcm_set_geometry(self.handle, grid, threads)

    def set_ghash_engine(self, engine: int) -> None:
        gcm_set_ghash_engine(self.handle, engine)

    def encrypt(self, iv, aad, pt, ct=None, stream=None):
        import torch
        if ct is None:
            ct = torch.empty_like(pt)
        return ct, gcm_encrypt(self.handle, iv, aad, pt, ct, stream)

    def decrypt_verify(self, iv, aad, ct, tag, pt=None, stream=None):
        import torch
        if pt is None:
            pt = torch.empty_like(ct)
        return gcm_decrypt_verify(self.handle, iv, aad, ct, pt, tag, stream), pt
