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
    assert len(gfc.EXPORTED_SYMBOLS) == 6


def test_argument_errors_without_gpu(lib_path):
    """Argument validation happens before any CUDA call."""
    import paper_2602_23067_b200 as pkg
    with pytest.raises(pkg.GcmError) as e:
        pkg.gcm_init(bytes(24))            # AES-192 is outside reading S1
    assert e.value.code == pkg.GCM_ERR_ARG
    L = ctypes.CDLL(lib_path)
    assert L.gcm_init(None, b"0" * 16, 128) == pkg.GCM_ERR_ARG
    assert L.gcm_encrypt(None, None, None, 0, None, 0, None, None, None) == pkg.GCM_ERR_ARG
    assert L.gfc_context_create(None, 0, 0) == pkg.GCM_ERR_ARG
    assert L.gfc_encrypt_frame(None, None, 0, None, None, 128, None, None, None) == pkg.GCM_ERR_ARG


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
