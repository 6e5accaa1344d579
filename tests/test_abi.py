"""The C-ABI library loads and exports every symbol include/gcm.h declares (no compute calls: no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2602_23067_b200 import build
    return build.build()


def declared_symbols(header="gcm.h", prefix="gcm_"):
    text = open(os.path.join(ROOT, "include", header)).read()
    return sorted(set(re.findall(r"GCM_API\s+[\w \*]+?\b(%s\w+)\s*\(" % prefix, text)))


def test_header_declares_the_boundary():
    names = declared_symbols()
    for must in ("gcm_init", "gcm_destroy", "gcm_encrypt", "gcm_decrypt_verify", "gcm_encrypt_batch",
                 "gcm_decrypt_verify_batch", "gcm_encrypt_async", "gcm_decrypt_verify_async"):
        assert must in names


def test_library_exports_every_declared_symbol(lib_path):
    L = ctypes.CDLL(lib_path)
    for name in declared_symbols() + declared_symbols("gfc.h", "gfc_"):
        assert hasattr(L, name), name
    L.gcm_version.restype = ctypes.c_char_p
    assert b"sm_100a" in L.gcm_version()


def test_binding_lists_the_same_symbols(lib_path):
    import paper_2602_23067_b200 as pkg
    assert sorted(pkg.EXPORTED_SYMBOLS) == declared_symbols()
    assert pkg.library_path() == lib_path
    from paper_2602_23067_b200 import gfc
    assert sorted(gfc.EXPORTED_SYMBOLS) == declared_symbols("gfc.h", "gfc_")
    assert len(gfc.EXPORTED_SYMBOLS) == 7


def test_argument_errors_without_gpu(lib_path):
    """Argument validation happens before any CUDA call."""
    import paper_2602_23067_b200 as pkg
    with pytest.raises(ValueError):
        pkg.gcm_init(bytes(24))            # AES-192 is outside reading S1
    with pytest.raises(ValueError):
        pkg.gcm_init(bytes(16), key_bits=256)      # key_bits must match the key (the C side would read 32 bytes)
    L = ctypes.CDLL(lib_path)
    assert L.gcm_init(None, b"0" * 16, 128) == pkg.GCM_ERR_ARG
    out = ctypes.c_void_p()
    assert L.gcm_init(ctypes.byref(out), b"0" * 24, 192) == pkg.GCM_ERR_ARG
    assert L.gcm_encrypt(None, None, None, 0, None, 0, None, None, None) == pkg.GCM_ERR_ARG
    assert L.gfc_context_create(None, 0, 0) == pkg.GCM_ERR_ARG
    assert L.gfc_encrypt_frame(None, None, 0, None, None, 128, None, None, None) == pkg.GCM_ERR_ARG


def test_binding_refuses_wrong_iv_and_tag_lengths(lib_path):
    """The C ABI takes `const uint8_t iv[12]` and reads exactly 12 bytes: an 11-byte IV would be read past its end, a
    16-byte one silently truncated (two IVs that differ in the last 4 bytes would collide; reading S5: 96-bit IVs
    only).  The binding refuses both in every entry point, before any pointer reaches C."""
    import paper_2602_23067_b200 as pkg
    ctx = 0xDEAD                          # never dereferenced: the length check comes first
    for bad in (bytes(11), bytes(16), b""):
        with pytest.raises(ValueError):
            pkg.gcm_encrypt(ctx, bad, None, None, None)
        with pytest.raises(ValueError):
            pkg.gcm_decrypt_verify(ctx, bad, None, None, None, bytes(16))
        with pytest.raises(ValueError):
            pkg.gcm_encrypt_async(ctx, bad, None, None, None, None)
        with pytest.raises(ValueError):
            pkg.gcm_decrypt_verify_async(ctx, bad, None, None, None, None, None)
        with pytest.raises(ValueError):
            pkg.gcm_encrypt_host(ctx, bad, None, None, None)
        with pytest.raises(ValueError):
            pkg.gcm_decrypt_verify_host(ctx, bad, None, None, None, bytes(16))
        with pytest.raises(ValueError):
            pkg.gcm_encrypt_batch([{"key": bytes(16), "iv": bad, "aad": None, "input": None, "output": None}])
    for bad_tag in (bytes(15), bytes(17)):
        with pytest.raises(ValueError):
            pkg.gcm_decrypt_verify(ctx, bytes(12), None, None, None, bad_tag)
        with pytest.raises(ValueError):
            pkg.gcm_decrypt_verify_host(ctx, bytes(12), None, None, None, bad_tag)


def test_no_cpu_fallback_in_product_path():
    """The product package never imports the oracle (checked textually)."""
    pkg_dir = os.path.join(ROOT, "paper_2602_23067_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "liboracle" not in text, f


def test_headers_are_plain_c(tmp_path):
    """The boundary is a C ABI: both headers must compile as C11 with no C++ and no CUDA or torch types."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    src = tmp_path / "use.c"
    src.write_text('#include "gcm.h"\n#include "gfc.h"\n'
                   "int main(void) { gcm_msg m; FitsOperationResult r; (void)m; (void)r;\n"
                   "  return (int)sizeof(m) + (int)sizeof(r) + GCM_ERR_AUTH + GFC_ERR_FORMAT + GCM_RATE_COUNT > 0 ? 0 : 1; }\n")
    subprocess.run([gcc, "-std=c11", "-Wall", "-Werror", "-pedantic", "-fsyntax-only", "-I", os.path.join(ROOT, "include"), str(src)],
                   check=True)
    for h in ("gcm.h", "gfc.h"):
        text = open(os.path.join(ROOT, "include", h)).read()
        assert "#include <cuda" not in text and "#include <torch" not in text and "at::Tensor" not in text, h
