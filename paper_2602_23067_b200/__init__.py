"""B200-native AES-GCM engine (arxiv/paper_2602_23067's hot path, re-designed for sm_100a).

The product is libb200gcm.so (csrc/, C ABI in include/gcm.h).  This package is only its Python
binding: same entry-point names, argument marshalling only.  There is no CPU fallback: the first use of any
name below loads `paper_2602_23067_b200.gcm`, which raises if the CUDA library has not been built
(`paper_2602_23067_b200.build` stays importable so that the library can be built first).
"""
_BINDING_NAMES = (
    "GCM_OK", "GCM_ERR_AUTH", "GCM_ERR_ARG", "GCM_ERR_LEN", "GCM_ERR_CUDA", "GCM_ERR_NOMEM", "GCM_ERR_BUSY", "GCM_PHASE_SLOTS",
    "GcmError", "GcmMsg", "Context", "gcm_version", "gcm_set_device", "gcm_last_cuda_error",
    "gcm_last_cuda_error_string", "gcm_init", "gcm_destroy", "gcm_set_geometry",
    "gcm_get_geometry", "gcm_set_ghash_engine", "gcm_get_ghash_engine", "GCM_GHASH_TABLE", "GCM_GHASH_TENSOR", "GCM_GHASH_AUTO", "TC2_AUTO_BYTES", "GHASH_TC_AUTO_BYTES", "gcm_get_hash_subkey", "gcm_encrypt", "gcm_decrypt_verify",
    "gcm_encrypt_async", "gcm_decrypt_verify_async", "gcm_ghash_async", "gcm_encrypt_host",
    "gcm_decrypt_verify_host", "gcm_decrypt_verify_host_strict", "gcm_set_phase_stamps", "gcm_encrypt_batch", "gcm_decrypt_verify_batch",
    "MsgBatch", "gcm_pack_msgs", "gcm_batch_release", "gcm_encrypt_batch_device", "gcm_decrypt_verify_batch_device", "gcm_pack_dmsgs", "gcm_debug_row_layout", "gcm_debug_plan_chunks", "gcm_debug_tc2_clock", "gcm_dmsg_dtype", "GCM_DMSG_BYTES", "gcm_measure_pipe_rates", "RATE_NAMES", "library_path", "EXPORTED_SYMBOLS",
)
__all__ = list(_BINDING_NAMES)


def __getattr__(name):
    if name in _BINDING_NAMES:
        from . import gcm as _gcm      # raises ImportError when libb200gcm.so is missing
        for n in _BINDING_NAMES:
            globals()[n] = getattr(_gcm, n)
        return globals()[name]
    raise AttributeError("module %r has no attribute %r" % (__name__, name))
