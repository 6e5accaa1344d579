"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the oracle tests, the GPU parity tests and bench.py.  It contains NO
AES / GHASH / GCM arithmetic -- only random bytes, FITS-style header text and FITS-shaped pixel
arrays -- so that the oracle and the CUDA path see the same bytes without sharing any of the
method's code.

The inputs stand in for the paper's real and synthetic FITS exposures (PAPER.md L297, L658,
Table A.7), which are not available here; AES-GCM cost does not depend on the data.
Generator: numpy.random.Generator(PCG64(seed)); draws in the fixed order key -> IV -> AAD -> payload.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List

import numpy as np

FITS_BLOCK = 2880  # bytes; FITS headers and data units are padded to multiples of this
SEEDS = {"C1": 1001, "C2": 1002, "C3": 1003, "C4": 1004, "C5": 1005}


@dataclass
class Message:
    key: bytes
    iv: bytes
    aad: np.ndarray      # uint8
    payload: np.ndarray  # uint8
    name: str = ""
    meta: dict = field(default_factory=dict)


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def _bytes(rng: np.random.Generator, n: int) -> np.ndarray:
    return rng.integers(0, 256, size=n, dtype=np.uint8)


def random_payload(rng: np.random.Generator, n: int) -> np.ndarray:
    """Uniform random uint8, generated 8 bytes at a time (fast enough for 4 GiB)."""
    words = rng.integers(0, 2 ** 64, size=(n + 7) // 8, dtype=np.uint64)
    return words.view(np.uint8)[:n]


# -------------------------------------------------------------------------------------------------
# FITS header block: 36 cards of 80 ASCII characters = 2880 bytes.
# Our own card formatter (astropy is not installed): keyword left-justified in columns 1-8,
# "= " in 9-10, value right-justified to column 30 for numbers / logicals, strings quoted from
# column 11; END card; blank padding.
# -------------------------------------------------------------------------------------------------
def _card(key: str, value=None, comment: str = "") -> str:
    if value is None:
        s = key
    else:
        if isinstance(value, bool):
            v = ("T" if value else "F").rjust(20)
        elif isinstance(value, int):
            v = str(value).rjust(20)
        elif isinstance(value, float):
            v = ("%.10G" % value).rjust(20)
        else:
            v = ("'%s'" % str(value).ljust(8)).ljust(20)
        s = "%-8s= %s" % (key, v)
        if comment:
            s += " / " + comment
    return s[:80].ljust(80)


def fits_header_block(rng: np.random.Generator, naxis1: int, naxis2: int, index: int = 0) -> np.ndarray:
    ra = float(rng.uniform(0.0, 360.0))
    dec = float(rng.uniform(-30.0, 60.0))
    scale = 0.4 / 3600.0
    cards = [
        _card("SIMPLE", True, "conforms to FITS standard"),
        _card("BITPIX", -32, "IEEE single precision floating point"),
        _card("NAXIS", 2, "number of array dimensions"),
        _card("NAXIS1", naxis1),
        _card("NAXIS2", naxis2),
        _card("EXTEND", True),
        _card("OBJECT", "FIELD%04d" % index, "synthetic field"),
        _card("TELESCOP", "SYNTH-1"),
        _card("INSTRUME", "SYNCAM"),
        _card("FILTER", "r"),
        _card("EXPTIME", float(rng.choice([30.0, 60.0, 120.0, 300.0])), "[s]"),
        _card("DATE-OBS", "2026-01-%02dT%02d:%02d:%02d" % (1 + int(rng.integers(0, 28)),
                                                          int(rng.integers(0, 24)),
                                                          int(rng.integers(0, 60)),
                                                          int(rng.integers(0, 60)))),
        _card("CTYPE1", "RA---TAN"),
        _card("CTYPE2", "DEC--TAN"),
        _card("CRVAL1", ra, "[deg]"),
        _card("CRVAL2", dec, "[deg]"),
        _card("CRPIX1", naxis1 / 2.0),
        _card("CRPIX2", naxis2 / 2.0),
        _card("CD1_1", -scale),
        _card("CD1_2", 0.0),
        _card("CD2_1", 0.0),
        _card("CD2_2", scale),
        _card("EQUINOX", 2000.0),
        _card("RADESYS", "ICRS"),
        _card("BUNIT", "adu"),
        _card("GAIN", 1.5, "[e-/adu]"),
        _card("RDNOISE", 4.2, "[e-]"),
        _card("AIRMASS", float(rng.uniform(1.0, 2.0))),
        _card("SEEING", 6.84 * 0.4, "[arcsec] FWHM"),
        _card("END"),
    ]
    text = "".join(cards).ljust(FITS_BLOCK)
    assert len(text) == FITS_BLOCK
    return np.frombuffer(text.encode("ascii"), dtype=np.uint8).copy()


def fits_image_payload(rng: np.random.Generator, ny: int, nx: int, n_sources: int = 200,
                       mean: float = 1000.0, sigma: float = 30.0) -> np.ndarray:
    """FITS-shaped data unit: big-endian float32 pixels (BITPIX = -32), Gaussian noise (mean,
    sigma) + seeded point sources (2-D Gaussians, FWHM ~ 6.84 px, peak log-uniform in [50, 20000])
    + 3 constant-valued (0.0) rectangles, zero-padded to a multiple of 2880 bytes."""
    img = rng.standard_normal(size=(ny, nx), dtype=np.float32) * np.float32(sigma) + np.float32(mean)
    s = 6.84 / 2.3548
    half = 12
    yy, xx = np.mgrid[-half: half + 1, -half: half + 1].astype(np.float32)
    for _ in range(n_sources):
        cy = int(rng.integers(half, max(half + 1, ny - half)))
        cx = int(rng.integers(half, max(half + 1, nx - half)))
        peak = float(np.exp(rng.uniform(np.log(50.0), np.log(20000.0))))
        dy, dx = float(rng.uniform(-0.5, 0.5)), float(rng.uniform(-0.5, 0.5))
        stamp = peak * np.exp(-((yy - dy) ** 2 + (xx - dx) ** 2) / (2 * s * s))
        y0, x0 = cy - half, cx - half
        if y0 >= 0 and x0 >= 0 and y0 + 2 * half + 1 <= ny and x0 + 2 * half + 1 <= nx:
            img[y0: y0 + 2 * half + 1, x0: x0 + 2 * half + 1] += stamp.astype(np.float32)
    for _ in range(3):
        h = int(rng.integers(max(1, ny // 16), max(2, ny // 4)))
        w = int(rng.integers(max(1, nx // 16), max(2, nx // 4)))
        y0 = int(rng.integers(0, ny - h + 1))
        x0 = int(rng.integers(0, nx - w + 1))
        img[y0: y0 + h, x0: x0 + w] = 0.0
    raw = img.astype(">f4").tobytes()
    pad = (-len(raw)) % FITS_BLOCK
    out = np.frombuffer(raw + b"\0" * pad, dtype=np.uint8)
    return out


# -------------------------------------------------------------------------------------------------
# The five configs.  `scale` arguments let the CPU-only tests use the same recipe at sizes the
# oracle finishes in seconds; the defaults are BASELINE.json's full sizes.
# -------------------------------------------------------------------------------------------------
def config_c1(payload_bytes: int = 1 << 20) -> Message:
    """C1: AES-128, 1 MiB uniform payload, 16-byte random AAD."""
    rng = _rng(SEEDS["C1"])
    key = _bytes(rng, 16).tobytes()
    iv = _bytes(rng, 12).tobytes()
    aad = _bytes(rng, 16)
    payload = random_payload(rng, payload_bytes)
    return Message(key, iv, aad, payload, "C1")


def config_c2(payload_bytes: int = 256 << 20) -> Message:
    """C2: AES-256, 256 MiB uniform payload, one 2880-byte FITS header block as AAD."""
    rng = _rng(SEEDS["C2"])
    key = _bytes(rng, 32).tobytes()
    iv = _bytes(rng, 12).tobytes()
    aad = fits_header_block(rng, 8192, 8192)
    payload = random_payload(rng, payload_bytes)
    return Message(key, iv, aad, payload, "C2")


def config_c3(n_images: int = 16, ny: int = 4096, nx: int = 4096, n_sources: int = 200) -> List[Message]:
    """C3: FITS-shaped batch, one AES-256 key, distinct IVs, per-image 2880-byte header as AAD
    (reading S14)."""
    rng0 = _rng(SEEDS["C3"])
    key = _bytes(rng0, 32).tobytes()
    msgs = []
    for i in range(n_images):
        rng = _rng(SEEDS["C3"] + 1 + i)
        iv = _bytes(rng, 12).tobytes()
        aad = fits_header_block(rng, nx, ny, index=i)
        payload = fits_image_payload(rng, ny, nx, n_sources=n_sources)
        msgs.append(Message(key, iv, aad, payload, "C3[%d]" % i))
    return msgs


def config_c4(n_messages: int = 10000, max_len: int = 65536, max_aad: int = 256) -> List[Message]:
    """C4: many short AES-128 messages, len ~ U{1..max_len}, AAD len ~ U{0..max_aad}, per-message
    random key and IV."""
    rng = _rng(SEEDS["C4"])
    lens = rng.integers(1, max_len + 1, size=n_messages)
    alens = rng.integers(0, max_aad + 1, size=n_messages)
    keys = _bytes(rng, 16 * n_messages).reshape(n_messages, 16)
    ivs = _bytes(rng, 12 * n_messages).reshape(n_messages, 12)
    aad_all = _bytes(rng, int(alens.sum()))
    pay_all = random_payload(rng, int(lens.sum()))
    msgs = []
    ao = po = 0
    for i in range(n_messages):
        a = aad_all[ao: ao + int(alens[i])]
        p = pay_all[po: po + int(lens[i])]
        ao += int(alens[i])
        po += int(lens[i])
        msgs.append(Message(keys[i].tobytes(), ivs[i].tobytes(), a, p, "C4[%d]" % i))
    return msgs


def config_c5(payload_bytes: int = 4 << 30, with_payload: bool = True) -> Message:
    """C5: AES-256, 4 GiB uniform payload, 2880-byte header AAD (reading S14), plus the seeded bit
    index of the tamper test in meta['flip_bit'].  with_payload=False returns key/IV/AAD only (the
    benchmark fills the payload on the device)."""
    rng = _rng(SEEDS["C5"])
    key = _bytes(rng, 32).tobytes()
    iv = _bytes(rng, 12).tobytes()
    aad = fits_header_block(rng, 32768, 32768)
    flip = int(rng.integers(0, 8 * payload_bytes))
    payload = random_payload(rng, payload_bytes) if with_payload else np.zeros(0, np.uint8)
    return Message(key, iv, aad, payload, "C5", {"flip_bit": flip, "payload_bytes": payload_bytes})


# -------------------------------------------------------------------------------------------------
# Whole FITS files for the authenticated-container path (section 3.2.2; the
# validation file of L245 is a 256 x 256 float32 image "with representative WCS metadata").
# -------------------------------------------------------------------------------------------------
@dataclass
class FitsFrame:
    fits: bytes          # a single-HDU FITS file: header block(s) + big-endian float32 data unit
    key_h: bytes         # Header Key
    key_d: bytes         # Data Key
    nonce_h: bytes       # 96-bit nonces (the paper draws them from the OS entropy pool, L137;
    nonce_d: bytes       # here they are seeded so that both implementations build the same bytes)
    ny: int = 0
    nx: int = 0


def fits_frame(seed: int = 2001, ny: int = 256, nx: int = 256, key_bytes: int = 16,
               n_sources: int = 20, extra_cards: int = 0) -> FitsFrame:
    """Draw order: key_h -> key_d -> nonce_h -> nonce_d -> header -> pixels.  extra_cards > 0 appends
    HISTORY cards so that the header spans several 2880-byte blocks."""
    rng = _rng(seed)
    key_h = _bytes(rng, key_bytes).tobytes()
    key_d = _bytes(rng, key_bytes).tobytes()
    nonce_h = _bytes(rng, 12).tobytes()
    nonce_d = _bytes(rng, 12).tobytes()
    hdr = fits_header_block(rng, nx, ny).tobytes()
    if extra_cards:
        text = hdr.decode("ascii")
        end = text.index("END".ljust(80))
        body = text[:end] + "".join(("HISTORY synthetic processing step %05d" % i).ljust(80) for i in range(extra_cards))
        body += "END".ljust(80)
        body += " " * ((-len(body)) % FITS_BLOCK)
        hdr = body.encode("ascii")
    data = fits_image_payload(rng, ny, nx, n_sources=n_sources).tobytes()
    return FitsFrame(hdr + data, key_h, key_d, nonce_h, nonce_d, ny, nx)
