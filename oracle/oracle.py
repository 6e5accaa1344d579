"""ctypes front end of the CPU oracle (oracle/gcm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It shares nothing with the CUDA path and never imports it.

All arithmetic lives in gcm_oracle.c (Eq. 1).  This
file only marshals arguments, and -- for the bounded cpu_baseline leg and the 4 GiB tag check --
spreads *independent* pieces over host threads:
  * CTR blocks are independent, so byte ranges go to threads as they are;
  * GHASH is the sequential Horner chain unless the caller asks for `ghash_segmented`, the derived
    identity documented (and pinned against Horner) next to orc_ghash_segment in the C file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gcm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_gcm.so")
_lock = threading.Lock()
_lib = None

AUTH_FAIL = 1


def build(force: bool = False) -> str:
    """Compile gcm_oracle.c with plain gcc -O2 (no intrinsics, no -march) into liboracle_gcm.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.run(
            ["gcc", "-std=c11", "-O2", "-Wall", "-Wextra", "-shared", "-fPIC", "-o", tmp, _SRC],
            check=True,
        )
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            L = ctypes.CDLL(build())
            u8p, u64, ci = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int
            L.orc_init.argtypes = []
            L.orc_init.restype = None
            L.orc_sbox_generate.argtypes = [u8p, u8p]
            L.orc_sbox_generate.restype = None
            L.orc_key_expand.argtypes = [u8p, ci, u8p]
            L.orc_key_expand.restype = ci
            L.orc_gf_mul.argtypes = [u8p, u8p, u8p]
            L.orc_gf_mul.restype = None
            L.orc_gf_pow.argtypes = [u8p, u64, u8p]
            L.orc_gf_pow.restype = None
            L.orc_ghash_update.argtypes = [u8p, u8p, u8p, u64]
            L.orc_ghash_update.restype = None
            L.orc_ghash.argtypes = [u8p, u8p, u64, u8p, u64, u8p]
            L.orc_ghash.restype = None
            L.orc_ghash_segment.argtypes = [u8p, u8p, u64, u64, u8p]
            L.orc_ghash_segment.restype = None
            L.orc_ctr_xor.argtypes = [u8p, ci, u8p, u64, u8p, u8p, u64]
            L.orc_ctr_xor.restype = ci
            L.orc_hash_subkey.argtypes = [u8p, ci, u8p]
            L.orc_hash_subkey.restype = ci
            L.orc_ek_j0.argtypes = [u8p, ci, u8p, u8p]
            L.orc_ek_j0.restype = ci
            L.orc_ecb_block.argtypes = [u8p, ci, u8p, u8p, ci]
            L.orc_ecb_block.restype = ci
            L.orc_gcm_encrypt.argtypes = [u8p, ci, u8p, u8p, u64, u8p, u64, u8p, u8p]
            L.orc_gcm_encrypt.restype = ci
            L.orc_gcm_decrypt_verify.argtypes = [u8p, ci, u8p, u8p, u64, u8p, u64, u8p, u8p]
            L.orc_gcm_decrypt_verify.restype = ci
            L.orc_init()
            _lib = L
    return _lib


# ---------------------------------------------------------------------------------------------
# marshalling helpers: everything crosses as contiguous uint8 numpy arrays
# ---------------------------------------------------------------------------------------------
def _arr(x) -> np.ndarray:
    if isinstance(x, np.ndarray):
        a = x
        if a.dtype != np.uint8:
            a = a.view(np.uint8)
        return np.ascontiguousarray(a).reshape(-1)
    return np.frombuffer(bytes(x), dtype=np.uint8)


def _ptr(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data) if a.size else ctypes.c_void_p(0)


def _key_bits(key) -> int:
    return 8 * len(_arr(key))


def sbox():
    s = np.zeros(256, np.uint8)
    inv = np.zeros(256, np.uint8)
    lib().orc_sbox_generate(_ptr(s), _ptr(inv))
    return s, inv


def key_expand(key) -> np.ndarray:
    """Round-key words w[0 .. 4(Nr+1)-1] as uint32 (FIPS-197 word = big-endian bytes)."""
    k = _arr(key)
    w = np.zeros(60, np.uint32)
    nr = lib().orc_key_expand(_ptr(k), 8 * k.size, ctypes.c_void_p(w.ctypes.data))
    if nr < 0:
        raise ValueError("key must be 16 or 32 bytes")
    return w[: 4 * (nr + 1)].copy()


def ecb_encrypt_block(key, block) -> bytes:
    k, b = _arr(key), _arr(block)
    out = np.zeros(16, np.uint8)
    if lib().orc_ecb_block(_ptr(k), 8 * k.size, _ptr(b), _ptr(out), 0) < 0:
        raise ValueError("key must be 16 or 32 bytes")
    return out.tobytes()


def ecb_decrypt_block(key, block) -> bytes:
    k, b = _arr(key), _arr(block)
    out = np.zeros(16, np.uint8)
    if lib().orc_ecb_block(_ptr(k), 8 * k.size, _ptr(b), _ptr(out), 1) < 0:
        raise ValueError("key must be 16 or 32 bytes")
    return out.tobytes()


def gf_mul(x, y) -> bytes:
    a, b = _arr(x), _arr(y)
    out = np.zeros(16, np.uint8)
    lib().orc_gf_mul(_ptr(a), _ptr(b), _ptr(out))
    return out.tobytes()


def gf_pow(h, e: int) -> bytes:
    a = _arr(h)
    out = np.zeros(16, np.uint8)
    lib().orc_gf_pow(_ptr(a), ctypes.c_uint64(e), _ptr(out))
    return out.tobytes()


def hash_subkey(key) -> bytes:
    k = _arr(key)
    out = np.zeros(16, np.uint8)
    if lib().orc_hash_subkey(_ptr(k), 8 * k.size, _ptr(out)) < 0:
        raise ValueError("key must be 16 or 32 bytes")
    return out.tobytes()


def ek_j0(key, iv) -> bytes:
    k, v = _arr(key), _arr(iv)
    assert v.size == 12
    out = np.zeros(16, np.uint8)
    if lib().orc_ek_j0(_ptr(k), 8 * k.size, _ptr(v), _ptr(out)) < 0:
        raise ValueError("key must be 16 or 32 bytes")
    return out.tobytes()


def ghash(h, aad, c) -> bytes:
    """GHASH_H(A || pad || C || pad || len64(A) || len64(C)), sequential Horner (Eq. 1)."""
    hh, a, cc = _arr(h), _arr(aad), _arr(c)
    out = np.zeros(16, np.uint8)
    lib().orc_ghash(_ptr(hh), _ptr(a), a.size, _ptr(cc), cc.size, _ptr(out))
    return out.tobytes()


def ghash_update(h, y, data) -> bytes:
    hh, d = _arr(h), _arr(data)
    yy = _arr(y).copy()
    lib().orc_ghash_update(_ptr(hh), _ptr(yy), _ptr(d), d.size)
    return yy.tobytes()


def ghash_segment(h, data, blocks_after: int) -> bytes:
    hh, d = _arr(h), _arr(data)
    out = np.zeros(16, np.uint8)
    lib().orc_ghash_segment(_ptr(hh), _ptr(d), d.size, ctypes.c_uint64(blocks_after), _ptr(out))
    return out.tobytes()


def ghash_segmented(h, aad, c, segment_blocks: int, threads: int = 1) -> bytes:
    """Same value as ghash(), computed by the segment identity (see orc_ghash_segment).

    The GHASH input is the block sequence A-blocks, C-blocks, length block.  It is cut into runs
    of `segment_blocks` blocks (never across the A/C boundary, because A and C are padded
    separately); each run is reduced by Horner and weighted by H^(blocks after it); the weighted
    values are XORed.  Runs are independent, so they may go to several host threads.
    """
    a, cc = _arr(aad), _arr(c)
    n_a = (a.size + 15) // 16
    n_c = (cc.size + 15) // 16
    jobs = []  # (array view, blocks_after)
    seg_bytes = 16 * segment_blocks
    for off in range(0, a.size, seg_bytes):
        piece = a[off: off + seg_bytes]
        done = off // 16 + (piece.size + 15) // 16
        jobs.append((piece, (n_a - done) + n_c + 1))
    for off in range(0, cc.size, seg_bytes):
        piece = cc[off: off + seg_bytes]
        done = off // 16 + (piece.size + 15) // 16
        jobs.append((piece, (n_c - done) + 1))
    lenblk = np.frombuffer(
        (8 * a.size).to_bytes(8, "big") + (8 * cc.size).to_bytes(8, "big"), dtype=np.uint8
    )
    jobs.append((lenblk, 0))

    def run(job):
        return np.frombuffer(ghash_segment(h, job[0], job[1]), dtype=np.uint8)

    if threads > 1:
        with ThreadPoolExecutor(threads) as ex:
            parts = list(ex.map(run, jobs))
    else:
        parts = [run(j) for j in jobs]
    acc = np.zeros(16, np.uint8)
    for p in parts:
        acc ^= p
    return acc.tobytes()


def ctr_xor(key, iv, data, first_block: int = 0, threads: int = 1) -> np.ndarray:
    """out = data ^ keystream, block g of the message using counter g + 2 (g counted from
    `first_block` at data[0]).  With threads > 1 the byte range is cut at block boundaries."""
    k, v, d = _arr(key), _arr(iv), _arr(data)
    assert v.size == 12
    out = np.empty_like(d)
    L = lib()

    def run(rng):
        lo, hi = rng
        if L.orc_ctr_xor(_ptr(k), 8 * k.size, _ptr(v), ctypes.c_uint64(first_block + lo // 16),
                         ctypes.c_void_p(d.ctypes.data + lo), ctypes.c_void_p(out.ctypes.data + lo),
                         ctypes.c_uint64(hi - lo)) < 0:
            raise ValueError("key must be 16 or 32 bytes")

    if d.size == 0:
        return out
    if threads <= 1:
        run((0, d.size))
    else:
        nblk = (d.size + 15) // 16
        per = (nblk + threads - 1) // threads * 16
        ranges = [(lo, min(lo + per, d.size)) for lo in range(0, d.size, per)]
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(run, ranges))
    return out


def keystream_block(key, iv, g: int) -> bytes:
    """E_K(IV || BE32(g + 2)): the keystream of payload block g, on its own."""
    return ctr_xor(key, iv, np.zeros(16, np.uint8), first_block=g).tobytes()


def gcm_encrypt(key, iv, aad, pt):
    """Returns (ciphertext as uint8 array, tag bytes).  Whole function, single thread, in C."""
    k, v, a, p = _arr(key), _arr(iv), _arr(aad), _arr(pt)
    assert v.size == 12
    ct = np.empty_like(p)
    tag = np.zeros(16, np.uint8)
    rc = lib().orc_gcm_encrypt(_ptr(k), 8 * k.size, _ptr(v), _ptr(a), a.size, _ptr(p), p.size,
                               _ptr(ct), _ptr(tag))
    if rc < 0:
        raise ValueError("orc_gcm_encrypt rc=%d" % rc)
    return ct, tag.tobytes()


def gcm_decrypt_verify(key, iv, aad, ct, tag):
    """Returns (status, plaintext array); status 0 = ok, 1 = authentication failure (zeros)."""
    k, v, a, c, t = _arr(key), _arr(iv), _arr(aad), _arr(ct), _arr(tag)
    assert v.size == 12 and t.size == 16
    pt = np.empty_like(c)
    rc = lib().orc_gcm_decrypt_verify(_ptr(k), 8 * k.size, _ptr(v), _ptr(a), a.size, _ptr(c),
                                      c.size, _ptr(pt), _ptr(t))
    if rc < 0:
        raise ValueError("orc_gcm_decrypt_verify rc=%d" % rc)
    return rc, pt


def gcm_encrypt_threaded(key, iv, aad, pt, threads: int, segment_blocks: int = 0):
    """The cpu_baseline / big-message form: CTR chunked over `threads`; GHASH sequential Horner
    when segment_blocks == 0 (the oracle proper), or by the pinned segment identity otherwise."""
    ct = ctr_xor(key, iv, pt, threads=threads)
    h = hash_subkey(key)
    s = ghash(h, aad, ct) if segment_blocks == 0 else ghash_segmented(h, aad, ct, segment_blocks, threads)
    e = ek_j0(key, iv)
    tag = bytes(x ^ y for x, y in zip(s, e))
    return ct, tag
