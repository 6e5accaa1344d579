"""Pins for oracle step 7 (GHASH; Eq. 1) and the segment identity behind the tree."""
import numpy as np
import pytest
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes
from cryptography.hazmat.primitives.ciphers.aead import AESGCM


def xor(a, b):
    return bytes(p ^ q for p, q in zip(a, b))


def lenblk(a, c):
    return (8 * a).to_bytes(8, "big") + (8 * c).to_bytes(8, "big")


def test_zero_and_single_block(oracle):
    rng = np.random.default_rng(3001)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    assert oracle.ghash(h, b"", b"") == bytes(16)                 # only the all-zero length block
    assert oracle.ghash_update(h, bytes(16), bytes(48)) == bytes(16)
    x = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    assert oracle.ghash_update(h, bytes(16), x) == oracle.gf_mul(x, h)
    # one ciphertext block: ((X.H) ^ L).H
    assert oracle.ghash(h, b"", x) == oracle.gf_mul(xor(oracle.gf_mul(x, h), lenblk(0, 16)), h)


def test_horner_equals_power_sum(oracle):
    """Y_N = sum_i X_i . H^(N-i+1): the closed form of Eq. 1, evaluated with gf_pow."""
    rng = np.random.default_rng(3002)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    for n in (1, 2, 3, 7, 20):
        data = rng.integers(0, 256, 16 * n, dtype=np.uint8).tobytes()
        acc = bytes(16)
        for i in range(n):
            acc = xor(acc, oracle.gf_mul(data[16 * i: 16 * i + 16], oracle.gf_pow(h, n - i)))
        assert oracle.ghash_update(h, bytes(16), data) == acc


def test_linearity_in_the_message(oracle):
    rng = np.random.default_rng(3003)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    for (a, c) in [(0, 16), (5, 37), (32, 160), (17, 1)]:
        a1 = rng.integers(0, 256, a, dtype=np.uint8).tobytes()
        a2 = rng.integers(0, 256, a, dtype=np.uint8).tobytes()
        c1 = rng.integers(0, 256, c, dtype=np.uint8).tobytes()
        c2 = rng.integers(0, 256, c, dtype=np.uint8).tobytes()
        g1 = oracle.ghash(h, a1, c1)
        g2 = oracle.ghash(h, a2, c2)
        g12 = oracle.ghash(h, xor(a1, a2), xor(c1, c2))
        g0 = oracle.ghash(h, bytes(a), bytes(c))       # carries the length block only
        # GHASH is affine in (A, C) at fixed lengths: the length block enters all four once
        assert xor(xor(g1, g2), g0) == g12


def test_partial_blocks_are_zero_padded_separately(oracle):
    rng = np.random.default_rng(3004)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    a = rng.integers(0, 256, 5, dtype=np.uint8).tobytes()
    c = rng.integers(0, 256, 21, dtype=np.uint8).tobytes()
    y = oracle.ghash_update(h, bytes(16), a + bytes(11))
    y = oracle.ghash_update(h, y, c + bytes(11))
    y = oracle.ghash_update(h, y, lenblk(5, 21))
    assert oracle.ghash(h, a, c) == y


def test_segmented_equals_horner_bruteforce(oracle):
    """Tree = Horner by brute force: every N from 0 to 320 blocks of C (with several AAD lengths,
    ragged tails) and every segment size from 1 to 9 plus the sizes the GPU geometry uses."""
    rng = np.random.default_rng(3005)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    data = rng.integers(0, 256, 16 * 330, dtype=np.uint8).tobytes()
    aad = rng.integers(0, 256, 100, dtype=np.uint8).tobytes()
    for n in list(range(0, 40)) + [63, 64, 65, 127, 128, 129, 255, 256, 257, 320]:
        for tail in (0, 1, 15):
            clen = max(0, 16 * n - tail)
            c = data[:clen]
            for alen in (0, 16, 33):
                ref = oracle.ghash(h, aad[:alen], c)
                for seg in (1, 2, 3, 4, 5, 7, 8, 9, 32, 128):
                    assert oracle.ghash_segmented(h, aad[:alen], c, seg) == ref, (n, tail, alen, seg)


def test_every_split_point(oracle):
    rng = np.random.default_rng(3006)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    n = 24
    data = rng.integers(0, 256, 16 * n, dtype=np.uint8).tobytes()
    ref = oracle.ghash_update(h, bytes(16), data)
    for cut in range(0, n + 1):
        left = oracle.ghash_segment(h, data[: 16 * cut], n - cut)
        right = oracle.ghash_segment(h, data[16 * cut:], 0)
        assert xor(left, right) == ref


def test_segmented_threads_match(oracle):
    rng = np.random.default_rng(3007)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    c = rng.integers(0, 256, 50001, dtype=np.uint8)
    a = rng.integers(0, 256, 2880, dtype=np.uint8)
    assert oracle.ghash_segmented(h, a, c, 100, threads=4) == oracle.ghash(h, a, c)


@pytest.mark.parametrize("klen", [16, 32])
def test_gmac_special_case_via_openssl(oracle, klen):
    """len = 0: T ^ E_K(J0) from OpenSSL must equal the oracle's GHASH_H(A || L) -- isolates GHASH
    (and H = E_K(0), J0) from CTR."""
    rng = np.random.default_rng(3100 + klen)
    for alen in list(range(0, 70)) + [255, 256, 257, 2880, 5000]:
        key = rng.integers(0, 256, klen, dtype=np.uint8).tobytes()
        iv = rng.integers(0, 256, 12, dtype=np.uint8).tobytes()
        aad = rng.integers(0, 256, alen, dtype=np.uint8).tobytes()
        tag = AESGCM(key).encrypt(iv, b"", aad)
        assert len(tag) == 16
        ecb = Cipher(algorithms.AES(key), modes.ECB()).encryptor()
        ek_j0 = ecb.update(iv + b"\x00\x00\x00\x01")
        h_lib = Cipher(algorithms.AES(key), modes.ECB()).encryptor().update(bytes(16))
        assert oracle.hash_subkey(key) == h_lib
        assert oracle.ek_j0(key, iv) == ek_j0
        assert oracle.ghash(h_lib, aad, b"") == xor(tag, ek_j0)
