"""GPU parity of the authenticated FITS container layer (include/gfc.h) against oracle/fits_container.py:
containers byte-identical for the same nonces, every access scenario of PAPER.md Table 2 (L261-L268) byte-identical,
DATASUM kernel against the oracle's sum, cross-decryption in both directions."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gfc():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2602_23067_b200 import gfc as g
    return g


@pytest.fixture(scope="module")
def F():
    from oracle import fits_container
    return fits_container


@pytest.fixture(scope="module")
def ctx(gfc):
    c = gfc.gfc_context_create(64 * 2880, 160 << 20)
    yield c
    gfc.gfc_context_destroy(c)


FRAMES = [
    dict(seed=2001, ny=256, nx=256, key_bytes=16, n_sources=20),                     # the paper's validation file, L245
    dict(seed=2002, ny=16, nx=24, key_bytes=32, n_sources=1, extra_cards=60),        # 3-block header, AES-256
    dict(seed=2003, ny=1, nx=1, key_bytes=16, n_sources=0),                          # one pixel
    dict(seed=2004, ny=1031, nx=977, key_bytes=32, n_sources=30, extra_cards=7),     # 4 MB, odd sizes
]


@pytest.mark.parametrize("spec", FRAMES, ids=lambda s: "seed%d" % s["seed"])
def test_container_bytes_match_oracle(gfc, F, ctx, spec):
    f = workloads.fits_frame(**spec)
    want = F.encrypt_frame(f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
    got = gfc.gfc_encrypt_frame(ctx, f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
    assert got.buffer_size == len(want)
    assert got.tobytes() == want


@pytest.mark.parametrize("spec", FRAMES[:2] + FRAMES[3:], ids=lambda s: "seed%d" % s["seed"])
def test_access_scenarios_match_oracle(gfc, F, ctx, spec):
    f = workloads.fits_frame(**spec)
    container = F.encrypt_frame(f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)    # oracle-written container
    other = bytes(len(f.key_h))
    for kh, kd in [(f.key_h, f.key_d), (f.key_h, None), (None, f.key_d), (None, None), (f.key_h, other), (other, f.key_d),
                   (other, other)]:
        want, warn = F.decrypt_frame(container, kh, kd)
        got = gfc.gfc_decrypt_frame(ctx, container, kh, kd)
        assert got.error_code == 0 and got.warning_code == warn, (kh is None, kd is None)
        assert got.tobytes() == want
    full = gfc.gfc_decrypt_frame(ctx, container, f.key_h, f.key_d)
    assert full.warning_code == gfc.GFC_FULL_ACCESS and full.tobytes() == f.fits      # bit-exact, L245


def test_tamper_matches_oracle(gfc, F, ctx):
    f = workloads.fits_frame(seed=2005, ny=64, nx=96, n_sources=4)
    c = F.encrypt_frame(f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)          # oracle-written; the CUDA path must agree
    assert gfc.gfc_encrypt_frame(ctx, f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d).tobytes() == c
    cases = []
    pos = c.index(b"ORIG_NA1=") + 29                      # last digit of the value
    cases.append(c[:pos] + bytes([c[pos] ^ 1]) + c[pos + 1:])
    pos = c.index(b"ENCHDR  = '") + 40
    cases.append(c[:pos] + (b"0" if c[pos:pos + 1] != b"0" else b"1") + c[pos + 1:])
    t = bytearray(c)
    t[-2880 * 3 + 1000] ^= 0x80
    cases.append(bytes(t))
    pos = c.index(b"AUTHTAGD= '") + 11
    cases.append(c[:pos] + (b"F" if c[pos:pos + 1] != b"F" else b"E") + c[pos + 1:])
    pos = c.index(b"NONCE_H = '") + 11
    cases.append(c[:pos] + (b"F" if c[pos:pos + 1] != b"F" else b"E") + c[pos + 1:])
    warns = []
    for t in cases:
        want, warn = F.decrypt_frame(t, f.key_h, f.key_d)
        got = gfc.gfc_decrypt_frame(ctx, t, f.key_h, f.key_d)
        assert got.warning_code == warn and got.tobytes() == want
        warns.append(warn)
    assert warns == [2, 1, 2, 2, 1]


def test_large_frame_multi_chunk(gfc, F, ctx):
    """A payload of several 64 MiB pipeline chunks with a ragged end: tag, DATASUM and CHECKSUM must still match."""
    rng = np.random.default_rng(7)
    f = workloads.fits_frame(seed=2006, ny=8, nx=8, n_sources=0)
    n = (64 << 20) + 2880 * 5 + 7                      # two pipeline chunks; not a multiple of 16 or of 2880
    payload = rng.integers(0, 256, n, dtype=np.uint8).tobytes()
    fits = f.fits[:2880] + payload                     # the container takes everything behind the header as payload (F2)
    want = F.encrypt_frame(fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
    got = gfc.gfc_encrypt_frame(ctx, fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
    assert got.buffer_size == len(want)
    assert np.array_equal(got.view(), np.frombuffer(want, np.uint8))
    back = gfc.gfc_decrypt_frame(ctx, want, f.key_h, f.key_d)
    assert back.warning_code == 0 and np.array_equal(back.view(), np.frombuffer(fits, np.uint8))
    assert back.header_ms > 0 and back.data_ms > 0


def test_datasum_kernel(gfc, F):
    import torch
    rng = np.random.default_rng(11)
    for n in [0, 1, 3, 4, 15, 16, 17, 2880, 2880 * 7 + 5, (1 << 20) + 13, (48 << 20) + 16 * 3 + 2]:
        a = rng.integers(0, 256, n, dtype=np.uint8)
        if n >= 2880:
            a[: n // 2] = 0xFF                               # long carry chains
        d = torch.from_numpy(a).cuda()
        pad = a.tobytes() + b"\0" * ((-n) % 4)
        assert gfc.gfc_datasum(d) == F.sum32(pad), n


def test_errors_and_random_nonces(gfc, F, ctx):
    f = workloads.fits_frame(seed=2007, ny=32, nx=32, n_sources=1)
    with pytest.raises(gfc.FrameError) as e:
        gfc.gfc_encrypt_frame(ctx, b"not a fits file".ljust(2880), f.key_h, f.key_d, f.nonce_h, f.nonce_d)
    assert e.value.code == gfc.GFC_ERR_FORMAT
    good = F.encrypt_frame(f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
    with pytest.raises(gfc.FrameError) as e:
        gfc.gfc_decrypt_frame(ctx, good[:-2880], f.key_h, f.key_d)
    assert e.value.code == gfc.GFC_ERR_FORMAT
    small = gfc.gfc_context_create(2880, 2880)
    try:
        with pytest.raises(gfc.FrameError) as e:
            gfc.gfc_encrypt_frame(small, f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
        assert e.value.code == gfc.GFC_ERR_CAPACITY
    finally:
        gfc.gfc_context_destroy(small)
    # nonces from the OS entropy pool (L137): two containers of the same file differ; with the nonces the library
    # drew (read back from the NONCE_H / NONCE_D cards, they are inputs) the oracle writes the same bytes
    a = gfc.gfc_encrypt_frame(ctx, f.fits, f.key_h, f.key_d).tobytes()
    b = gfc.gfc_encrypt_frame(ctx, f.fits, f.key_h, f.key_d).tobytes()
    assert a != b
    for c in (a, b):
        nh = bytes.fromhex(c[c.index(b"NONCE_H = '") + 11:][:24].decode())
        nd = bytes.fromhex(c[c.index(b"NONCE_D = '") + 11:][:24].decode())
        assert nh != f.nonce_h and nd != f.nonce_d and nh != nd
        assert c == F.encrypt_frame(f.fits, f.key_h, f.key_d, nh, nd)
        back = gfc.gfc_decrypt_frame(ctx, c, f.key_h, f.key_d)
        assert back.warning_code == 0 and back.tobytes() == f.fits
