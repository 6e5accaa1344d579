"""Full-size pins of the oracle forms that carry the GPU parity checks at C2 / C3 / C5 size.

tests/test_gpu_full_configs.py compares the GPU with `oracle.ctr_xor(..., threads=N)` and with GHASH by
weighted segments (`orc_ghash_segment`: Horner over a 1 MiB segment times H^(blocks after it), exponents up
to 2^28).  That blocking is the oracle's own, so it is pinned here, at the sizes it is used at, against an
implementation that shares nothing with it: the installed OpenSSL's streaming AES-GCM
(`Cipher(AES, GCM(iv))`, chunked `update_into`, "Whole GCM" row) -- and against the
oracle's own plain Horner chain (Eq. 1) at full C2 size.

A wrong power in the segment weights, a CTR chunk boundary off by a block, a counter that wraps early or a
length block with swapped halves all change the tag or the ciphertext here.
"""
import os

import numpy as np
import pytest
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes

import workloads

THREADS = os.cpu_count() or 1
SEG_BLOCKS = 1 << 16          # the segment size tests/test_gpu_full_configs.py uses (1 MiB)


def openssl_streaming_gcm(key, iv, aad, pt: np.ndarray, chunk: int = 1 << 30):
    """AES-GCM of `pt` through OpenSSL's incremental interface in `chunk`-byte updates (the one-shot AESGCM API
    stops below 2^31 bytes).  Returns (ciphertext array, tag)."""
    enc = Cipher(algorithms.AES(bytes(key)), modes.GCM(bytes(iv))).encryptor()
    enc.authenticate_additional_data(bytes(aad))
    out = np.empty(pt.size + 15, np.uint8)
    done = 0
    for off in range(0, pt.size, chunk):
        piece = pt[off: off + chunk]
        done += enc.update_into(memoryview(piece), memoryview(out)[done: done + piece.size + 15])
    tail = enc.finalize()
    assert tail == b"" and done == pt.size
    return out[:pt.size], enc.tag


def test_config_c2_full_size_against_streaming_openssl(oracle):
    """C2 as BASELINE.json states it (AES-256, 256 MiB, 2880-byte AAD): the threaded CTR + segmented GHASH form
    equals OpenSSL byte for byte, and the segmented GHASH equals the plain sequential Horner chain."""
    m = workloads.config_c2()
    assert m.payload.size == 256 << 20 and m.aad.size == 2880 and len(m.key) == 32
    ct, tag = oracle.gcm_encrypt_threaded(m.key, m.iv, m.aad, m.payload, threads=THREADS, segment_blocks=SEG_BLOCKS)
    ref_ct, ref_tag = openssl_streaming_gcm(m.key, m.iv, m.aad, m.payload, chunk=100 << 20)
    assert np.array_equal(ct, ref_ct)
    assert tag == ref_tag
    # Eq. 1 as written (one thread, no blocking) over the same 16,777,216 + 180 + 1 blocks
    h = oracle.hash_subkey(m.key)
    s_horner = oracle.ghash(h, m.aad, ct)
    assert s_horner == oracle.ghash_segmented(h, m.aad, ct, SEG_BLOCKS, THREADS)
    assert tag == bytes(x ^ y for x, y in zip(s_horner, oracle.ek_j0(m.key, m.iv)))


def test_window_walk_of_the_gpu_tests_against_streaming_openssl(oracle):
    """The exact walk `oracle_check_device_message` does (128 MiB windows, ctr_xor with first_block, 1 MiB
    segments weighted by H^(blocks after), AAD and length block as their own segments) on a 160 MiB + 5-byte
    message: two windows, the second ragged, a partial last block."""
    from concurrent.futures import ThreadPoolExecutor
    n = (160 << 20) + 5
    m = workloads.config_c5(payload_bytes=n)
    aad = m.aad[:777]
    window = 128 << 20
    n_c = (n + 15) // 16
    h = oracle.hash_subkey(m.key)
    acc = np.frombuffer(oracle.ghash_segment(h, aad, n_c + 1), np.uint8).copy()
    ct = np.empty(n, np.uint8)
    for off in range(0, n, window):
        hi = min(n, off + window)
        ct[off:hi] = oracle.ctr_xor(m.key, m.iv, m.payload[off:hi], first_block=off // 16, threads=THREADS)
        jobs = []
        for s in range(off, hi, 16 * SEG_BLOCKS):
            piece = ct[s: min(hi, s + 16 * SEG_BLOCKS)]
            jobs.append((piece, n_c - (s // 16 + (piece.size + 15) // 16) + 1))
        with ThreadPoolExecutor(THREADS) as ex:
            for part in ex.map(lambda j: oracle.ghash_segment(h, j[0], j[1]), jobs):
                acc ^= np.frombuffer(part, np.uint8)
    lenblk = (8 * aad.size).to_bytes(8, "big") + (8 * n).to_bytes(8, "big")
    acc ^= np.frombuffer(oracle.ghash_segment(h, lenblk, 0), np.uint8)
    tag = bytes(x ^ y for x, y in zip(acc.tobytes(), oracle.ek_j0(m.key, m.iv)))
    ref_ct, ref_tag = openssl_streaming_gcm(m.key, m.iv, aad, m.payload, chunk=64 << 20)
    assert np.array_equal(ct, ref_ct)
    assert tag == ref_tag


@pytest.mark.slow
def test_config_c5_size_plus_ragged_tail_against_streaming_openssl(oracle):
    """C5 size and beyond: 4 GiB + 13 bytes (block indices above 2^28, byte offsets above 2^32, a partial last
    block), AES-256, 2880-byte AAD; OpenSSL in 1 GiB updates.  About a minute and 13 GiB of host memory."""
    psutil = pytest.importorskip("psutil")
    if psutil.virtual_memory().available < 16 << 30:
        pytest.skip("needs 16 GiB of free host memory")
    n = (4 << 30) + 13
    m = workloads.config_c5(payload_bytes=n)
    assert m.payload.size == n
    ct, tag = oracle.gcm_encrypt_threaded(m.key, m.iv, m.aad, m.payload, threads=THREADS, segment_blocks=SEG_BLOCKS)
    ref_ct, ref_tag = openssl_streaming_gcm(m.key, m.iv, m.aad, m.payload, chunk=1 << 30)
    assert tag == ref_tag
    for off in range(0, n, 256 << 20):                       # windowed compare keeps the temporaries small
        assert np.array_equal(ct[off: off + (256 << 20)], ref_ct[off: off + (256 << 20)]), off
