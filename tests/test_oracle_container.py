"""Pins of the container oracle (oracle/fits_container.py) against what the paper and the FITS standard fix:
the layout of PAPER.md L115-L125, the AAD formula of L151-L155 (with the paper's own example '-32'), the four
access scenarios of Table 2 (L261-L268) / L245, the checksum invariant of the convention cited at L135, and the
installed OpenSSL as an independent decryptor of ENCHDR and of the BINTABLE blob.  CPU only."""
import numpy as np
import pytest
from cryptography.exceptions import InvalidTag
from cryptography.hazmat.primitives.ciphers.aead import AESGCM

import workloads
from oracle import fits_container as F


# ---- an independent, minimal reading of the FITS structure (no code shared with the oracle) -------------------
def walk_hdus(buf: bytes):
    """Yields (dict keyword -> raw value text, header offset, data offset, data length) per HDU."""
    assert len(buf) % 2880 == 0, "FITS files are a whole number of 2880-byte blocks"
    pos = 0
    out = []
    while pos < len(buf):
        kw, order = {}, []
        p = pos
        last_key = None
        while True:
            card = buf[p:p + 80].decode("ascii")          # must be pure ASCII
            assert all(32 <= ord(ch) < 127 for ch in card)
            p += 80
            key = card[:8].rstrip()
            if key == "END":
                assert card[8:].strip() == ""
                break
            if key == "CONTINUE":
                text = card[10:].strip()
                assert text.startswith("'") and last_key is not None and kw[last_key].endswith("&")
                kw[last_key] = kw[last_key][:-1] + text[1:text.rindex("'")]
                continue
            assert card[8:10] == "= ", card
            v = card[10:].split("/")[0].strip() if "'" not in card[10:] else card[10:].strip()
            if v.startswith("'"):
                v = v[1:v.rindex("'")].rstrip()
            kw[key] = v
            order.append(key)
            last_key = key
        hdr_end = pos + ((p - pos + 2879) // 2880) * 2880
        assert buf[p:hdr_end].strip(b" ") == b"", "header padding must be blanks"
        naxis = int(kw["NAXIS"])
        n = abs(int(kw["BITPIX"])) // 8
        for i in range(1, naxis + 1):
            n *= int(kw["NAXIS%d" % i])
        if naxis == 0:
            n = 0
        n *= int(kw.get("GCOUNT", 1))
        n += int(kw.get("PCOUNT", 0))
        out.append((kw, order, pos, hdr_end, n))
        pos = hdr_end + (n + 2879) // 2880 * 2880
    assert pos == len(buf)
    return out


def ones_complement_sum_slow(b: bytes) -> int:
    s = 0
    for i in range(0, len(b), 4):
        s += int.from_bytes(b[i:i + 4], "big")
        s = (s & 0xFFFFFFFF) + (s >> 32)
    return s


@pytest.fixture(scope="module")
def frame():
    return workloads.fits_frame(seed=2001, ny=48, nx=40, n_sources=3)


@pytest.fixture(scope="module")
def container(frame):
    return F.encrypt_frame(frame.fits, frame.key_h, frame.key_d, frame.nonce_h, frame.nonce_d)


def test_structure_two_hdus(frame, container):
    hdus = walk_hdus(container)
    assert len(hdus) == 2
    kw0, order0, _, _, n0 = hdus[0]
    assert order0[:3] == ["SIMPLE", "BITPIX", "NAXIS"] and kw0["SIMPLE"] == "T" and kw0["NAXIS"] == "0" and n0 == 0
    assert kw0["EXTEND"] == "T"
    assert bytes.fromhex(kw0["NONCE_H"]) == frame.nonce_h and bytes.fromhex(kw0["NONCE_D"]) == frame.nonce_d
    assert len(bytes.fromhex(kw0["AUTHTAGH"])) == 16 and len(bytes.fromhex(kw0["AUTHTAGD"])) == 16
    # footnote 3 (L127): abbreviated ORIG_* names, values of the original header in plain text
    assert (kw0["ORIG_BPX"], kw0["ORIG_NAX"], kw0["ORIG_NA1"], kw0["ORIG_NA2"]) == ("-32", "2", "40", "48")
    assert all(len(k) <= 8 for k in order0)
    kw1, order1, _, d1, n1 = hdus[1]
    assert order1[:8] == ["XTENSION", "BITPIX", "NAXIS", "NAXIS1", "NAXIS2", "PCOUNT", "GCOUNT", "TFIELDS"]
    assert kw1["XTENSION"] == "BINTABLE" and kw1["NAXIS2"] == "1" and kw1["TFIELDS"] == "1"
    payload_len = len(frame.fits) - 2880
    assert n1 == payload_len and kw1["TFORM1"] == "%dB" % payload_len          # L125: TFORM = '<N>B'
    assert len(bytes.fromhex(kw0["ENCHDR"])) == 2880                             # the complete original header


def test_checksum_invariant(container):
    """FITS checksum convention: with CHECKSUM in place the 1's-complement sum of every HDU is -0, DATASUM is the
    decimal sum of the data unit, and the 16 characters are alphanumeric."""
    hdus = walk_hdus(container)
    for i, (kw, _, h0, d0, n) in enumerate(hdus):
        end = d0 + (n + 2879) // 2880 * 2880
        assert ones_complement_sum_slow(container[h0:end]) == 0xFFFFFFFF
        assert int(kw["DATASUM"]) == ones_complement_sum_slow(container[d0:end])
        assert len(kw["CHECKSUM"]) == 16 and kw["CHECKSUM"].isalnum()
    # a corrupted byte breaks the sum
    bad = bytearray(container)
    bad[-5] ^= 0x10
    assert ones_complement_sum_slow(bytes(bad[hdus[1][2]:])) != 0xFFFFFFFF


def test_checksum_encode_is_its_own_inverse_under_the_sum():
    """The 16 characters, placed at byte offset 11 mod 4 = 3 as in the card, must add the encoded value (minus the
    sum of sixteen '0' characters) to the record's sum: this is what the convention defines."""
    rng = np.random.default_rng(5)
    for v in [0, 1, 0xFFFFFFFF, 0x80000000, 0x12345678] + [int(x) for x in rng.integers(0, 2 ** 32, 200)]:
        s = F.checksum_encode(v)
        assert len(s) == 16 and s.isalnum()
        rec = (b"CHECKSUM= '" + s.encode() + b"'").ljust(80)
        zero = (b"CHECKSUM= '" + b"0" * 16 + b"'").ljust(80)
        a, z = ones_complement_sum_slow(rec), ones_complement_sum_slow(zero)
        # a = z (+) v in 1's-complement arithmetic
        t = z + v
        t = (t & 0xFFFFFFFF) + (t >> 32)
        assert a % 0xFFFFFFFF == t % 0xFFFFFFFF, hex(v)


def test_aad_formula_papers_example():
    """L155: 'the integer -32 becomes the byte sequence "-32"'; L151-L153: NONCE_D first, then the keywords."""
    n = bytes(range(12))
    assert F.aad_data(n, -32, 2, [4096, 2048]) == n + b"-32" + b"2" + b"4096" + b"2048"
    assert F.aad_data(n, 16, 0, []) == n + b"160"


def test_openssl_opens_both_messages(frame, container):
    """Independent decryptor: OpenSSL must open ENCHDR with (Header Key, NONCE_H, AAD = NONCE_H) and the blob with
    (Data Key, NONCE_D, AAD = NONCE_D || '-32' '2' '40' '48'), and must refuse with a changed AAD."""
    hdus = walk_hdus(container)
    kw0 = hdus[0][0]
    ct_h = bytes.fromhex(kw0["ENCHDR"])
    hdr = AESGCM(frame.key_h).decrypt(frame.nonce_h, ct_h + bytes.fromhex(kw0["AUTHTAGH"]), frame.nonce_h)
    assert hdr == frame.fits[:2880]
    _, _, _, d1, n1 = hdus[1]
    blob = container[d1:d1 + n1]
    aad = frame.nonce_d + b"-3224048"
    pix = AESGCM(frame.key_d).decrypt(frame.nonce_d, blob + bytes.fromhex(kw0["AUTHTAGD"]), aad)
    assert pix == frame.fits[2880:]
    with pytest.raises(InvalidTag):
        AESGCM(frame.key_d).decrypt(frame.nonce_d, blob + bytes.fromhex(kw0["AUTHTAGD"]), frame.nonce_d + b"-3224084")


def test_four_access_scenarios(frame, container):
    """Table 2 (L261-L268) and L245: full access is bit-exact; header key only -> zero-filled payload; data key only
    -> minimal header + pixels; wrong keys behave like missing keys; every output is valid FITS."""
    other = bytes(16)
    out, w = F.decrypt_frame(container, frame.key_h, frame.key_d)
    assert w == 0 and out == frame.fits
    for kd in (None, other):
        out, w = F.decrypt_frame(container, frame.key_h, kd)
        assert w == F.WARN_PAYLOAD_SUPPRESSED and out[:2880] == frame.fits[:2880] and not any(out[2880:])
        assert len(out) == len(frame.fits) and len(walk_hdus(out)) == 1
    for kh in (None, other):
        out, w = F.decrypt_frame(container, kh, frame.key_d)
        assert w == F.WARN_HEADER_FALLBACK and out[2880:] == frame.fits[2880:]
        (kw, order, _, _, n), = walk_hdus(out)
        assert order == ["SIMPLE", "BITPIX", "NAXIS", "NAXIS1", "NAXIS2"]
        assert (kw["BITPIX"], kw["NAXIS1"], kw["NAXIS2"]) == ("-32", "40", "48")
    out, w = F.decrypt_frame(container, None, None)
    assert w == 3 and not any(out[2880:]) and len(walk_hdus(out)) == 1


def _replace_card_value(container: bytes, key: str, old: str, new: str) -> bytes:
    k = key.ljust(8).encode()
    for pos in range(0, 2880 * 4, 80):
        if container[pos:pos + 8] == k:
            card = container[pos:pos + 80]
            assert old.encode() in card
            return container[:pos] + card.replace(old.encode(), new.encode(), 1) + container[pos + 80:]
    raise AssertionError(key)


def test_tamper_is_compartmentalised(frame, container):
    """L157 / Figure 2: tampering with a plaintext ORIG_* value breaks AUTHTAG_D (payload suppressed) but not the
    header; tampering with ENCHDR breaks AUTHTAG_H only; a flipped ciphertext bit suppresses the payload."""
    t = _replace_card_value(container, "ORIG_NA1", "40", "41")
    out, w = F.decrypt_frame(t, frame.key_h, frame.key_d)
    assert w == F.WARN_PAYLOAD_SUPPRESSED and out[:2880] == frame.fits[:2880] and not any(out[2880:])
    pos = container.index(b"ENCHDR  = '") + 11
    ch = container[pos:pos + 1]
    t = container[:pos] + (b"0" if ch != b"0" else b"1") + container[pos + 1:]
    out, w = F.decrypt_frame(t, frame.key_h, frame.key_d)
    assert w == F.WARN_HEADER_FALLBACK and out[2880:] == frame.fits[2880:]
    t = bytearray(container)
    t[-2880 * 2 + 17] ^= 0x04
    out, w = F.decrypt_frame(bytes(t), frame.key_h, frame.key_d)
    assert w == F.WARN_PAYLOAD_SUPPRESSED and not any(out[2880:])
    t = _replace_card_value(container, "NONCE_D", frame.nonce_d.hex().upper()[:2], "%02X" % (frame.nonce_d[0] ^ 1))
    out, w = F.decrypt_frame(t, frame.key_h, frame.key_d)
    assert w == F.WARN_PAYLOAD_SUPPRESSED


def test_multi_block_header_and_aes256():
    f = workloads.fits_frame(seed=2002, ny=16, nx=24, key_bytes=32, n_sources=1, extra_cards=60)
    assert f.fits.index(b"END".ljust(80)) > 2880            # header spans several blocks
    c = F.encrypt_frame(f.fits, f.key_h, f.key_d, f.nonce_h, f.nonce_d)
    hdus = walk_hdus(c)
    assert len(bytes.fromhex(hdus[0][0]["ENCHDR"])) == 3 * 2880
    out, w = F.decrypt_frame(c, f.key_h, f.key_d)
    assert w == 0 and out == f.fits


def test_malformed_containers_are_errors(container):
    with pytest.raises(F.ContainerError):
        F.decrypt_frame(container[:2880], b"k" * 16, b"k" * 16)
    with pytest.raises(F.ContainerError):
        F.decrypt_frame(_replace_card_value(container, "NONCE_H", "'", "'ZZ"), b"k" * 16, b"k" * 16)
    with pytest.raises(F.ContainerError):
        F.decrypt_frame(container[:-2880], b"k" * 16, b"k" * 16)
