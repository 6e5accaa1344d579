/*
 * gfc.h -- C ABI of the authenticated FITS container layer of libb200gcm.so.
 *
 * Names and result structure follow the paper's Table 1 and Listing 1 (L483-L538):
 * gfc_context_create / gfc_decrypt_frame / gfc_context_destroy and FitsOperationResult {data_buffer,
 * buffer_size, error_code, warning_code, error_message}; gfc_encrypt_frame is the writer the paper describes
 * in section 3.2.2 (L113-L125) without naming its entry point.
 *
 * What a frame call does (section 3.2.2-3.2.3, section 3.3.2, section 4.2
 * L237-L245; the readings F1-F12 of DESIGN.md section 11 fill what the paper leaves open):
 *   - the original single-file FITS image is split into a two-HDU container: HDU 0 is a metadata-only
 *     primary HDU holding NONCE_H, NONCE_D, AUTHTAGH, AUTHTAGD, the plaintext structural keywords
 *     ORIG_BPX / ORIG_NAX / ORIG_NAn and ENCHDR = the complete original header encrypted with the Header
 *     Key; HDU 1 is a one-row, one-column BINTABLE (TFORM1 = '<N>B') holding the payload encrypted with
 *     the Data Key.  Both HDUs carry CHECKSUM / DATASUM.
 *   - the data message's AAD is NONCE_D || ASCII-decimal(ORIG_BITPIX) || ASCII-decimal(ORIG_NAXIS) || ...
 *     (L151-L155), so the plaintext structural keywords are bound to the pixels.
 *   - the header message travels on the context's streamH and the data message on streamD, concurrently
 *     (L211-L217); the data message is chunked through pinned memory (H2D -> fused AES-GCM kernel ->
 *     DATASUM kernel -> D2H).  All AES / GHASH / tag / compare / DATASUM arithmetic runs in CUDA kernels;
 *     the host only parses and formats 80-character cards.
 *   - decryption never fails on a missing or wrong key: a missing / wrong Header Key gives a minimal header
 *     rebuilt from ORIG_* (warning 1), a missing / wrong Data Key or any tampering with the ciphertext, the
 *     tag, NONCE_D or ORIG_* gives a zero-filled payload (warning 2); both give 3.
 *
 * All pointers are HOST pointers.  `fits` / `container` may be pageable or pinned (pinned gives full PCIe
 * rate).  A context serves one call at a time.  There is no CPU fallback: without a CUDA device
 * gfc_context_create returns GCM_ERR_CUDA.
 */
#ifndef B200_GFC_H
#define B200_GFC_H

#include <stdint.h>
#include "gcm.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gfc_context gfc_context; /* opaque: two CUDA streams, pinned buffers, cached key contexts */

enum {
    GFC_ERR_FORMAT   = -5,  /* not a FITS file / not a container this library wrote                       */
    GFC_ERR_CAPACITY = -6   /* header or payload larger than the sizes given to gfc_context_create         */
    /* other negative codes are the GCM_ERR_* of gcm.h */
};

enum {                       /* FitsOperationResult.warning_code                        */
    GFC_FULL_ACCESS        = 0,
    GFC_HEADER_FALLBACK    = 1,
    GFC_PAYLOAD_SUPPRESSED = 2   /* 3 = both (reading F10)                                                  */
};

typedef struct {
    uint8_t *data_buffer;    /* host (pinned), OWNED BY THE CONTEXT: valid until the next call on it or its  */
                             /* destruction.  encrypt: the container; decrypt: a FITS file ready for a reader */
    uint64_t buffer_size;
    int      error_code;     /* 0 success (then check warning_code); < 0 system / format error               */
    int      warning_code;   /* decrypt only                                                                  */
    float    header_ms;      /* device time of the header message on streamH (H2D + kernel + D2H)            */
    float    data_ms;        /* device time of the data message pipeline on streamD                           */
    char     error_message[128];
} FitsOperationResult;

/*
 * gfc_context_create -- "Initializes session: pre-allocates pinned memory and CUDA streams" (L170-L171,
 * L233): streamH, streamD, a pinned result buffer sized for max_header_bytes + max_data_bytes plus the
 * container's own cards, device staging.  Returns GCM_OK / GCM_ERR_ARG / GCM_ERR_NOMEM / GCM_ERR_CUDA.
 */
GCM_API int gfc_context_create(gfc_context **out, uint64_t max_header_bytes, uint64_t max_data_bytes);

/* Zeroises cached key contexts and staging buffers, frees everything.  NULL is ignored. */
GCM_API void gfc_context_destroy(gfc_context *ctx);

/*
 * gfc_encrypt_frame -- writes the container for one FITS file.
 *   fits, fits_len   the original file: primary header (n x 2880 bytes, END card) followed by the payload
 *                    (everything behind the header, reading F2)
 *   key_h, key_d     Header Key and Data Key, key_bits / 8 bytes each (128 or 256)
 *   nonce_h, nonce_d 12 bytes each; NULL = drawn from the OS entropy pool (/dev/urandom, L137)
 *   res              out; data_buffer / buffer_size = the container
 * Returns res->error_code.
 */
GCM_API int gfc_encrypt_frame(gfc_context *ctx, const uint8_t *fits, uint64_t fits_len,
                              const uint8_t *key_h, const uint8_t *key_d, int key_bits,
                              const uint8_t *nonce_h, const uint8_t *nonce_d, FitsOperationResult *res);

/*
 * gfc_decrypt_frame -- "Decrypts and authenticates a FITS frame" (L172-L174).
 *   key_h, key_d     NULL = key not provisioned (Table 2)
 *   res              out; data_buffer / buffer_size = a syntactically valid FITS file in every access
 *                    scenario (L245); warning_code says which one
 * Returns res->error_code (0 also for partial access: "never crash the read", L245).
 */
GCM_API int gfc_decrypt_frame(gfc_context *ctx, const uint8_t *container, uint64_t container_len,
                              const uint8_t *key_h, const uint8_t *key_d, int key_bits,
                              FitsOperationResult *res);

/*
 * gfc_datasum -- the FITS DATASUM of a device-resident buffer (1's-complement sum of big-endian 32-bit
 * words, missing tail bytes read as zero; the convention the paper cites at L135), computed by the
 * library's HBM-bound reduction kernel.  d_data: device, len bytes, 16-byte aligned.  sum: host, out.
 * Synchronises `cuda_stream`.
 */
GCM_API int gfc_datasum(const void *d_data, uint64_t len, uint32_t *sum, void *cuda_stream);

/*
 * Asynchronous form for device-timed measurement and for summing a data unit piece by piece: adds the
 * sum of d_data[0, len) to *d_acc (device, one uint64 the caller zeroes first; pieces must start at
 * multiples of 4 bytes of the data unit).  No synchronisation.  The DATASUM is the accumulator folded
 * with end-around carry: s = (s & 0xFFFFFFFF) + (s >> 32) until s < 2^32.
 */
GCM_API int gfc_datasum_async(const void *d_data, uint64_t len, void *d_acc, void *cuda_stream);

/*
 * gfc_datasum_noalloc -- the DATASUM of gfc_datasum for callers that cannot allocate device memory.
 *
 * gfc_datasum calls cudaMalloc and cudaFree for its accumulator on every call.  That rules it out (a) in a
 * process where something else already holds all of the GPU's memory (a framework's caching allocator, a
 * serving engine's pre-reserved pools: a raw cudaMalloc fails there) and (b) in a latency-sensitive loop that
 * runs beside other streams, because cudaMalloc / cudaFree may wait for the whole device.  This entry point
 * calls neither, nor any other allocating routine: its scratch is a 128.25 KiB array that is part of the
 * library's device image, so every GPU the library is used on holds those 128.25 KiB until the process exits.
 *
 *   d_data       device, len bytes, 16-byte aligned (may be NULL when len = 0)
 *   len          at most GFC_DATASUM_NOALLOC_MAX_BYTES (4 GiB: the array holds one partial sum per 256 KiB
 *                tile, 16384 of them); a longer buffer returns GCM_ERR_LEN and enqueues nothing -- sum it in
 *                pieces with gfc_datasum_async instead
 *   d_sum        device, out: one uint32, 4-byte aligned, the caller's own memory; written by the kernel
 *   cuda_stream  the work (an 8-byte memset of the scratch's counter + one kernel) is enqueued here; the call
 *                does not synchronise: read *d_sum after the stream has reached that point
 *
 * The data must live on the calling thread's current device.  The first call on each device looks up the
 * scratch's device address (and makes the CUDA runtime load the library's module there if it has not yet):
 * make that call once at start-up, outside any stream capture and outside the latency-critical part.
 * All calls on one device share the one array: two calls whose kernels may run at the same time (two streams
 * with no ordering between them, two host threads) corrupt each other's sums.  Calls that follow each other on
 * one stream, or that are ordered by events, are safe; nothing has to be cleared between them.
 * Returns GCM_OK / GCM_ERR_ARG (NULL or misaligned pointer) / GCM_ERR_LEN / GCM_ERR_CUDA.
 */
#define GFC_DATASUM_NOALLOC_MAX_BYTES (1ull << 32)
GCM_API int gfc_datasum_noalloc(const void *d_data, uint64_t len, uint32_t *d_sum, void *cuda_stream);

#ifdef __cplusplus
}
#endif

#endif /* B200_GFC_H */
