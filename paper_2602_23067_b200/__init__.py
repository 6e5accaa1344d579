"""B200-native AES-GCM engine (arxiv/paper_2602_23067's hot path, re-designed for sm_100a).

The product is libb200gcm.so (csrc/, C ABI in include/gcm.h).  This package is only its Python
binding: same entry-point names, argument marshalling only.  There is no CPU fallback: importing
`paper_2602_23067_b200.gcm` raises if the CUDA library has not been built.
"""
from .gcm import (  # noqa: F401
    GCM_OK, GCM_ERR_AUTH, GCM_ERR_ARG, GCM_ERR_LEN, GCM_ERR_CUDA, GCM_ERR_NOMEM,
    GcmError, GcmMsg, Context,
    gcm_version, gcm_set_device, gcm_last_cuda_error, gcm_last_cuda_error_string,
    gcm_init, gcm_destroy, gcm_set_geometry, gcm_get_geometry, gcm_get_hash_subkey,
    gcm_encrypt, gcm_decrypt_verify, gcm_encrypt_async, gcm_decrypt_verify_async, gcm_ghash_async,
    gcm_encrypt_host, gcm_decrypt_verify_host,
    gcm_encrypt_batch, gcm_decrypt_verify_batch, gcm_batch_release,
    library_path, EXPORTED_SYMBOLS,
)
