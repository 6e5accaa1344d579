"""Pins for oracle steps 1-3 (S-box, key expansion, block cipher).  SURVEY.md 8(c) pin table."""
import numpy as np
import pytest
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes


def test_sbox_is_a_permutation_with_closed_forms(oracle):
    s, inv = oracle.sbox()
    assert sorted(s.tolist()) == list(range(256))
    assert s[0] == 0x63                      # S(0) = Aff(0) = the affine constant c
    idx = np.arange(256, dtype=np.uint8)
    assert not np.any(s == idx)              # no fixed point
    assert not np.any(s == (idx ^ 0xFF))     # no opposite fixed point
    assert np.array_equal(inv[s], idx)       # inverse table really inverts
    # the affine map is invertible and 0x63 only enters as a constant: S(a)^S(b) never 0 for a != b
    assert len(set((s ^ s[0]).tolist())) == 256


def test_sbox_inverse_of_one_is_affine_of_one(oracle):
    # 1 is its own inverse in GF(2^8), so S(1) = Aff(1): bits 0,4,5,6,7 of input 1 -> rows that see a_0
    # b_i = a_i ^ a_{i+4} ^ a_{i+5} ^ a_{i+6} ^ a_{i+7} ^ c_i with a = 0x01 sets b_0,b_1,b_2,b_3,b_4
    # (those i for which one of i, i+4..i+7 is 0 mod 8) = 0x1F, then ^ 0x63
    s, _ = oracle.sbox()
    assert s[1] == (0x1F ^ 0x63)


@pytest.mark.parametrize("klen", [16, 32])
def test_round_key_count_and_first_words(oracle, klen):
    rng = np.random.default_rng(7 + klen)
    key = rng.integers(0, 256, klen, dtype=np.uint8).tobytes()
    w = oracle.key_expand(key)
    assert len(w) == (44 if klen == 16 else 60)
    for i in range(klen // 4):
        assert int(w[i]) == int.from_bytes(key[4 * i: 4 * i + 4], "big")


def test_bad_key_size_rejected(oracle):
    with pytest.raises(ValueError):
        oracle.key_expand(bytes(24))        # AES-192 is outside reading S1
    with pytest.raises(ValueError):
        oracle.ecb_encrypt_block(bytes(15), bytes(16))


@pytest.mark.parametrize("klen", [16, 32])
def test_inverse_cipher_roundtrip(oracle, klen):
    rng = np.random.default_rng(11 + klen)
    for _ in range(200):
        key = rng.integers(0, 256, klen, dtype=np.uint8).tobytes()
        blk = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
        ct = oracle.ecb_encrypt_block(key, blk)
        assert ct != blk
        assert oracle.ecb_decrypt_block(key, ct) == blk


@pytest.mark.parametrize("klen", [16, 32])
def test_block_cipher_matches_openssl_ecb(oracle, klen):
    """Library special case: one AES-ECB block via the installed OpenSSL on 10^4 seeded pairs.
    Any key-schedule error (incl. the extra SubWord at i mod 8 = 4 for AES-256) changes every output."""
    rng = np.random.default_rng(100 + klen)
    keys = rng.integers(0, 256, (10000, klen), dtype=np.uint8)
    blks = rng.integers(0, 256, (10000, 16), dtype=np.uint8)
    # structured corner inputs as well
    keys[0] = 0; blks[0] = 0
    keys[1] = 0xFF; blks[1] = 0xFF
    keys[2] = np.arange(klen); blks[2] = np.arange(16) * 17
    for i in range(10000):
        k = keys[i].tobytes()
        b = blks[i].tobytes()
        enc = Cipher(algorithms.AES(k), modes.ECB()).encryptor()
        assert oracle.ecb_encrypt_block(k, b) == enc.update(b), i
