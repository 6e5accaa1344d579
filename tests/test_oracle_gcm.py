"""Pins for oracle steps 4-5, 8-9 (CTR, tag, decrypt-verify) and the whole function."""
import numpy as np
import pytest
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes
from cryptography.hazmat.primitives.ciphers.aead import AESGCM

import workloads


def _mk(rng, klen, n, a):
    key = rng.integers(0, 256, klen, dtype=np.uint8).tobytes()
    iv = rng.integers(0, 256, 12, dtype=np.uint8).tobytes()
    aad = rng.integers(0, 256, a, dtype=np.uint8).tobytes()
    pt = rng.integers(0, 256, n, dtype=np.uint8).tobytes()
    return key, iv, aad, pt


@pytest.mark.parametrize("klen", [16, 32])
def test_whole_gcm_matches_openssl_small_grid(oracle, klen):
    """Library special case = the whole function: all (len, a) in [0,100] x [0,40]."""
    rng = np.random.default_rng(4000 + klen)
    for n in range(0, 101):
        for a in range(0, 41):
            key, iv, aad, pt = _mk(rng, klen, n, a)
            ct, tag = oracle.gcm_encrypt(key, iv, aad, pt)
            assert ct.tobytes() + tag == AESGCM(key).encrypt(iv, pt, aad), (n, a)


@pytest.mark.parametrize("klen", [16, 32])
def test_whole_gcm_matches_openssl_boundaries(oracle, klen):
    """Sizes straddling 16-byte, 512-block-row and CTA-stride boundaries of the GPU geometry."""
    rng = np.random.default_rng(4100 + klen)
    sizes = [255, 256, 257, 4095, 4096, 4097, 8191, 8192, 8193, 16 * 512 - 1, 16 * 512 + 1,
             65535, 65536, 65537, 16 * 1024 * 3 + 5]
    for n in sizes:
        for a in (0, 1, 16, 2880):
            key, iv, aad, pt = _mk(rng, klen, n, a)
            ct, tag = oracle.gcm_encrypt(key, iv, aad, pt)
            assert ct.tobytes() + tag == AESGCM(key).encrypt(iv, pt, aad), (n, a)


def test_streaming_openssl_on_config_c1(oracle):
    """C1 at full size (1 MiB) against OpenSSL's streaming GCM; also the threaded oracle form
    (CTR chunked across threads, GHASH by the segment identity) against the plain one."""
    m = workloads.config_c1()
    ct, tag = oracle.gcm_encrypt(m.key, m.iv, m.aad, m.payload)
    enc = Cipher(algorithms.AES(m.key), modes.GCM(m.iv)).encryptor()
    enc.authenticate_additional_data(m.aad.tobytes())
    ref = b""
    pt = m.payload.tobytes()
    for off in range(0, len(pt), 100000):
        ref += enc.update(pt[off: off + 100000])
    ref += enc.finalize()
    assert ct.tobytes() == ref
    assert tag == enc.tag
    ct2, tag2 = oracle.gcm_encrypt_threaded(m.key, m.iv, m.aad, m.payload, threads=4, segment_blocks=4096)
    assert np.array_equal(ct, ct2) and tag2 == tag
    ct3, tag3 = oracle.gcm_encrypt_threaded(m.key, m.iv, m.aad, m.payload, threads=3, segment_blocks=0)
    assert np.array_equal(ct, ct3) and tag3 == tag


@pytest.mark.parametrize("klen", [16, 32])
def test_closed_form_empty_message(oracle, klen):
    """a = len = 0  =>  T = E_K(J0) exactly (reading S6)."""
    rng = np.random.default_rng(4200 + klen)
    key, iv, _, _ = _mk(rng, klen, 0, 0)
    ct, tag = oracle.gcm_encrypt(key, iv, b"", b"")
    assert ct.size == 0
    assert tag == oracle.ek_j0(key, iv)
    ecb = Cipher(algorithms.AES(key), modes.ECB()).encryptor()
    assert tag == ecb.update(iv + b"\x00\x00\x00\x01")


@pytest.mark.parametrize("klen", [16, 32])
def test_ctr_properties(oracle, klen):
    rng = np.random.default_rng(4300 + klen)
    key, iv, _, pt = _mk(rng, klen, 1000, 0)
    pt2 = rng.integers(0, 256, 1000, dtype=np.uint8).tobytes()
    c1 = oracle.ctr_xor(key, iv, pt)
    c2 = oracle.ctr_xor(key, iv, pt2)
    ks = oracle.ctr_xor(key, iv, bytes(1000))
    # keystream independent of P
    assert np.array_equal(c1 ^ np.frombuffer(pt, np.uint8), ks)
    assert np.array_equal(c2 ^ np.frombuffer(pt2, np.uint8), ks)
    # prefix property
    for n in (1, 15, 16, 17, 999):
        assert np.array_equal(oracle.ctr_xor(key, iv, pt[:n]), c1[:n])
    # block g of the keystream is ECB(IV || BE32(g + 2)) from the library (reading S2)
    for g in (0, 1, 2, 61):
        ecb = Cipher(algorithms.AES(key), modes.ECB()).encryptor()
        assert ks[16 * g: 16 * g + 16].tobytes() == ecb.update(iv + (g + 2).to_bytes(4, "big"))
        assert oracle.keystream_block(key, iv, g) == ks[16 * g: 16 * g + 16].tobytes()
    # geometry-agnostic: any chunking / thread count gives the same bytes
    for th in (2, 3, 8):
        assert np.array_equal(oracle.ctr_xor(key, iv, pt, threads=th), c1)
    # a far block index (beyond 2^28) through first_block
    g = (1 << 28) + 12345
    ecb = Cipher(algorithms.AES(key), modes.ECB()).encryptor()
    assert oracle.keystream_block(key, iv, g) == ecb.update(iv + (g + 2).to_bytes(4, "big"))


@pytest.mark.parametrize("klen", [16, 32])
def test_roundtrip_and_tamper(oracle, klen):
    rng = np.random.default_rng(4400 + klen)
    for (n, a) in [(0, 0), (0, 9), (1, 0), (16, 16), (257, 33), (5000, 2880)]:
        key, iv, aad, pt = _mk(rng, klen, n, a)
        ct, tag = oracle.gcm_encrypt(key, iv, aad, pt)
        rc, back = oracle.gcm_decrypt_verify(key, iv, aad, ct, tag)
        assert rc == 0 and back.tobytes() == pt
        # OpenSSL accepts what the oracle produced
        assert AESGCM(key).decrypt(iv, ct.tobytes() + tag, aad) == pt

        def rejected(k=key, v=iv, A=aad, C=ct, T=tag):
            rc, out = oracle.gcm_decrypt_verify(k, v, A, C, T)
            return rc == oracle.AUTH_FAIL and not out.any()

        for bit in range(0, 128, 13):                         # tag bits
            t = bytearray(tag); t[bit // 8] ^= 1 << (bit % 8)
            assert rejected(T=bytes(t))
        if n:
            for pos in sorted({0, n // 2, n - 1}):            # ciphertext bits
                c = ct.copy(); c[pos] ^= 0x10
                assert rejected(C=c)
            assert rejected(C=ct[:-1])                        # length change
        if a:
            A = bytearray(aad); A[a // 2] ^= 0x01
            assert rejected(A=bytes(A))
            assert rejected(A=aad[:-1])
        v = bytearray(iv); v[5] ^= 0x80
        assert rejected(v=bytes(v))
        k = bytearray(key); k[0] ^= 1
        assert rejected(k=bytes(k))


def test_length_limit(oracle):
    import ctypes
    L = oracle.lib()
    key = bytes(16); iv = bytes(12); tag = (ctypes.c_uint8 * 16)()
    rc = L.orc_gcm_encrypt(key, 128, iv, None, 0, None, (1 << 36) - 31, None, tag)
    assert rc == -2


def test_scaled_configs_against_openssl(oracle):
    """The five configs' recipes at CPU-sized scale, whole function vs OpenSSL."""
    msgs = [workloads.config_c1(1 << 14), workloads.config_c2(100003)]
    msgs += workloads.config_c3(n_images=2, ny=96, nx=80, n_sources=5)
    msgs += workloads.config_c4(n_messages=40, max_len=3000)
    msgs += [workloads.config_c5(70001)]
    for m in msgs:
        ct, tag = oracle.gcm_encrypt(m.key, m.iv, m.aad, m.payload)
        assert ct.tobytes() + tag == AESGCM(m.key).encrypt(m.iv, m.payload.tobytes(), m.aad.tobytes()), m.name
