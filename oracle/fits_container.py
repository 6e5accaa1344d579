"""ORACLE (test infrastructure, not product code) for the authenticated FITS container of
PAPER.md section 3.2.2-3.2.3 (L113-L157), the dual-key access scenarios of section 4.2 / Table 2
(L237-L245, L261-L268) and the FITS checksum convention the paper cites (L135).

Plain Python + numpy on top of the plain-C GCM oracle (oracle.py); slow and obvious on purpose.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this.  It shares no
code with paper_2602_23067_b200/ (the product's container code is C++ in csrc/gfc_frame.cu).

Where the paper is silent the readings F1-F12 of DESIGN.md section 11 are taken; each is marked below.

Container layout (L115-L125, Figure 2):
  HDU 0  metadata-only primary HDU (NAXIS = 0): NONCE_H, NONCE_D, AUTHTAGH, AUTHTAGD, ORIG_BPX, ORIG_NAX,
         ORIG_NA1.., ENCHDR (the complete original header, encrypted with the Header Key), CHECKSUM, DATASUM
  HDU 1  BINTABLE, one row, one column TFORM1 = '<N>B': the payload encrypted with the Data Key
"""
from __future__ import annotations

import numpy as np

from . import oracle as O

BLOCK = 2880
CARD = 80

WARN_FULL = 0              # L181-L183: 0 full access, 1 header fallback, 2 payload suppressed
WARN_HEADER_FALLBACK = 1
WARN_PAYLOAD_SUPPRESSED = 2   # both at once: 3 (reading F10)


class ContainerError(ValueError):
    pass


# ---- FITS cards (FITS standard 4.0 section 4.2, fixed format) -------------------------------------
def card_logical(key: str, v: bool) -> bytes:
    return ("%-8s= %20s" % (key, "T" if v else "F")).ljust(CARD).encode("ascii")


def card_int(key: str, v: int) -> bytes:
    return ("%-8s= %20d" % (key, v)).ljust(CARD).encode("ascii")


def card_str(key: str, s: str) -> bytes:
    assert "'" not in s and len(s) <= 68
    return ("%-8s= '%s'" % (key, s.ljust(8))).ljust(CARD).encode("ascii")


def cards_long_str(key: str, s: str) -> list:
    """OGIP long-string convention: 67 characters + '&' per card, CONTINUE cards carry the rest (F4)."""
    pieces = [s[i:i + 67] for i in range(0, len(s), 67)] or [""]
    out = []
    for i, p in enumerate(pieces):
        text = p + ("&" if i + 1 < len(pieces) else "")
        if i == 0:
            out.append(("%-8s= '%s'" % (key, text.ljust(8))).ljust(CARD).encode("ascii"))
        else:
            out.append(("CONTINUE  '%s'" % text).ljust(CARD).encode("ascii"))
    return out


def pad_block(b: bytes, fill: bytes) -> bytes:
    r = (-len(b)) % BLOCK
    return b + fill * r


def parse_header(buf: bytes, off: int = 0):
    """Cards of the header that starts at `off`: returns (list of 80-byte cards up to END, header length)."""
    cards = []
    pos = off
    while True:
        if pos + CARD > len(buf):
            raise ContainerError("header without END")
        c = buf[pos:pos + CARD]
        pos += CARD
        if c[:8] == b"END     " and c[8:].strip() == b"":
            break
        cards.append(c)
    hlen = ((pos - off) + BLOCK - 1) // BLOCK * BLOCK
    if off + hlen > len(buf):
        raise ContainerError("truncated header block")
    return cards, hlen


def card_value(cards, key: str):
    """Value field of the first card with that keyword: int, bool or str (long strings joined)."""
    k = key.ljust(8).encode("ascii")
    for i, c in enumerate(cards):
        if c[:8] == k and c[8:10] == b"= ":
            v = c[10:].decode("ascii")
            if v.lstrip().startswith("'"):
                s = _quoted(v)
                j = i + 1
                while s.endswith("&") and j < len(cards) and cards[j][:10] == b"CONTINUE  ":
                    s = s[:-1] + _quoted(cards[j][10:].decode("ascii"))
                    j += 1
                return s
            v = v.split("/")[0].strip()
            if v in ("T", "F"):
                return v == "T"
            return int(v)
    return None


def _quoted(v: str) -> str:
    a = v.index("'")
    b = v.index("'", a + 1)          # values written here never contain quotes
    return v[a + 1:b].rstrip(" ")


# ---- FITS checksum (Seaman 1995; FITS standard 4.0 appendix J), cited by the paper at L135 --------
def sum32(data: bytes, start: int = 0) -> int:
    """1's-complement sum of the bytes as big-endian 32-bit words (length a multiple of 4)."""
    assert len(data) % 4 == 0
    s = start + int(np.frombuffer(data, dtype=">u4").astype(np.uint64).sum())
    while s >> 32:
        s = (s & 0xFFFFFFFF) + (s >> 32)       # end-around carry
    return s


def checksum_encode(value: int) -> str:
    """The 16-character ASCII encoding of a 32-bit value (appendix J.2): each byte is split into four
    characters around '0' that sum to it, punctuation is avoided by +1/-1 on pairs, and the string is
    rotated right by one so that it lands 4-byte aligned in columns 12-27 of the card."""
    exclude = set(range(0x3A, 0x41)) | set(range(0x5B, 0x61))
    asc = [0] * 16
    for i in range(4):
        byte = (value >> (24 - 8 * i)) & 0xFF
        q, r = divmod(byte, 4)
        ch = [q + 0x30 + r, q + 0x30, q + 0x30, q + 0x30]
        again = True
        while again:
            again = False
            for j in (0, 2):
                if ch[j] in exclude or ch[j + 1] in exclude:
                    ch[j] += 1
                    ch[j + 1] -= 1
                    again = True
        for j in range(4):
            asc[4 * j + i] = ch[j]
    return "".join(chr(asc[(i + 15) % 16]) for i in range(16))


def finish_hdu(header_cards: list, data: bytes) -> bytes:
    """Header (cards + DATASUM + CHECKSUM + END, blank-padded) followed by the data (zero-padded),
    with the two checksum keywords set so that the 1's-complement sum of the whole HDU is -0."""
    data_p = pad_block(data, b"\0")
    dsum = sum32(data_p)
    cards = list(header_cards) + [card_str("DATASUM", str(dsum)), card_str("CHECKSUM", "0" * 16)]
    hdr = pad_block(b"".join(cards) + b"END".ljust(CARD), b" ")
    total = sum32(hdr, dsum)
    cards[-1] = card_str("CHECKSUM", checksum_encode(~total & 0xFFFFFFFF))
    hdr = pad_block(b"".join(cards) + b"END".ljust(CARD), b" ")
    return hdr + data_p


# ---- the container ---------------------------------------------------------------------------------
def orig_keywords(cards):
    """BITPIX, NAXIS, NAXIS1..NAXISn of the original primary header (L121, footnote 3)."""
    bitpix = card_value(cards, "BITPIX")
    naxis = card_value(cards, "NAXIS")
    if not isinstance(bitpix, int) or not isinstance(naxis, int) or isinstance(bitpix, bool) or not 0 <= naxis <= 9:
        raise ContainerError("BITPIX / NAXIS missing")
    dims = []
    for i in range(1, naxis + 1):
        d = card_value(cards, "NAXIS%d" % i)
        if not isinstance(d, int) or isinstance(d, bool) or d < 0:
            raise ContainerError("NAXIS%d missing" % i)
        dims.append(d)
    return bitpix, naxis, dims


def aad_data(nonce_d: bytes, bitpix: int, naxis: int, dims) -> bytes:
    """L151-L155: NONCE_D || Serialize(ORIG_BITPIX) || Serialize(ORIG_NAXIS) || Serialize(ORIG_NAXISn)...,
    Serialize = strict ASCII decimal ('-32'), plain concatenation (F6)."""
    return nonce_d + b"".join(str(v).encode("ascii") for v in [bitpix, naxis] + list(dims))


def encrypt_frame(fits: bytes, key_h: bytes, key_d: bytes, nonce_h: bytes, nonce_d: bytes) -> bytes:
    cards, hlen = parse_header(fits)
    bitpix, naxis, dims = orig_keywords(cards)
    header = fits[:hlen]
    payload = fits[hlen:]                                 # F2: everything behind the primary header
    ct_h, tag_h = O.gcm_encrypt(key_h, nonce_h, nonce_h, header)           # F7: AAD_H = NONCE_H
    ct_d, tag_d = O.gcm_encrypt(key_d, nonce_d, aad_data(nonce_d, bitpix, naxis, dims), payload)
    c0 = [card_logical("SIMPLE", True), card_int("BITPIX", 8), card_int("NAXIS", 0), card_logical("EXTEND", True),
          card_str("LONGSTRN", "OGIP 1.0"),
          card_str("NONCE_H", nonce_h.hex().upper()), card_str("NONCE_D", nonce_d.hex().upper()),
          card_str("AUTHTAGH", tag_h.hex().upper()), card_str("AUTHTAGD", tag_d.hex().upper()),
          card_int("ORIG_BPX", bitpix), card_int("ORIG_NAX", naxis)]
    c0 += [card_int("ORIG_NA%d" % (i + 1), d) for i, d in enumerate(dims)]
    c0 += cards_long_str("ENCHDR", ct_h.tobytes().hex().upper())
    n = len(payload)
    c1 = [card_str("XTENSION", "BINTABLE"), card_int("BITPIX", 8), card_int("NAXIS", 2), card_int("NAXIS1", n),
          card_int("NAXIS2", 1), card_int("PCOUNT", 0), card_int("GCOUNT", 1), card_int("TFIELDS", 1),
          card_str("TTYPE1", "ENCDATA"), card_str("TFORM1", "%dB" % n), card_str("EXTNAME", "ENCDATA")]
    return finish_hdu(c0, b"") + finish_hdu(c1, ct_d.tobytes())


def fallback_header(bitpix: int, naxis: int, dims) -> bytes:
    """L241: 'a structurally valid, minimal FITS header' from the plaintext ORIG_* keywords (F9)."""
    cards = [card_logical("SIMPLE", True), card_int("BITPIX", bitpix), card_int("NAXIS", naxis)]
    cards += [card_int("NAXIS%d" % (i + 1), d) for i, d in enumerate(dims)]
    return pad_block(b"".join(cards) + b"END".ljust(CARD), b" ")


def decrypt_frame(container: bytes, key_h, key_d):
    """Returns (fits bytes, warning code).  key_h / key_d = None: key not provisioned (Table 2)."""
    c0, h0len = parse_header(container)
    if card_value(c0, "NAXIS") != 0:
        raise ContainerError("HDU 0 is not metadata-only")
    try:
        nonce_h = bytes.fromhex(card_value(c0, "NONCE_H"))
        nonce_d = bytes.fromhex(card_value(c0, "NONCE_D"))
        tag_h = bytes.fromhex(card_value(c0, "AUTHTAGH"))
        tag_d = bytes.fromhex(card_value(c0, "AUTHTAGD"))
        ct_h = bytes.fromhex(card_value(c0, "ENCHDR"))
    except (TypeError, ValueError):
        raise ContainerError("bad envelope keyword")
    if len(nonce_h) != 12 or len(nonce_d) != 12 or len(tag_h) != 16 or len(tag_d) != 16:
        raise ContainerError("bad envelope keyword length")
    bitpix, naxis = card_value(c0, "ORIG_BPX"), card_value(c0, "ORIG_NAX")
    if not isinstance(bitpix, int) or not isinstance(naxis, int) or not 0 <= naxis <= 9:
        raise ContainerError("ORIG_* missing")
    dims = [card_value(c0, "ORIG_NA%d" % (i + 1)) for i in range(naxis)]
    if any(not isinstance(d, int) for d in dims):
        raise ContainerError("ORIG_NAn missing")
    c1, h1len = parse_header(container, h0len)
    n = card_value(c1, "NAXIS1")
    if card_value(c1, "XTENSION") != "BINTABLE" or not isinstance(n, int) or n < 0:
        raise ContainerError("HDU 1 is not the data container")
    d_off = h0len + h1len
    if d_off + n > len(container):
        raise ContainerError("truncated payload")
    ct_d = container[d_off:d_off + n]

    warning = 0
    header = None
    if key_h is not None:
        rc, pt = O.gcm_decrypt_verify(key_h, nonce_h, nonce_h, ct_h, tag_h)
        if rc == 0:
            header = pt.tobytes()
    if header is None:                                            # L241: header fallback
        header = fallback_header(bitpix, naxis, dims)
        warning |= WARN_HEADER_FALLBACK
    payload = None
    if key_d is not None:
        rc, pt = O.gcm_decrypt_verify(key_d, nonce_d, aad_data(nonce_d, bitpix, naxis, dims), ct_d, tag_d)
        if rc == 0:
            payload = pt.tobytes()
    if payload is None:                                           # L243: payload suppression (zero-fill)
        payload = b"\0" * n
        warning |= WARN_PAYLOAD_SUPPRESSED
    return header + payload, warning
