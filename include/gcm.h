/*
 * gcm.h -- C ABI of the B200-native AES-GCM engine (libb200gcm.so).
 *
 * The boundary follows the NIST SP 800-38D problem statement (the paper adopts it by reference,
 * PAPER.md L111, L137, L255) and SURVEY.md section 8(b).  The hot path behind it is the one the
 * paper's contribution targets: AES-CTR keystream XORed into the payload, fused with a GHASH over
 * A || C || len computed as a parallel reduction with precomputed powers of H instead of the serial
 * recurrence Y_i = (Y_{i-1} xor X_i) . H (Eq. 1; L272-L286, sections 5.2.1-5.2.2).
 *
 * Conventions
 *   - "host" pointers are ordinary CPU memory; "device" pointers are CUDA device memory on the
 *     context's device (e.g. the data_ptr() of a torch uint8 tensor).  The library never allocates
 *     or frees caller data.  A gcm_ctx owns its own device tables and scratch.
 *   - Return codes follow the paper's Table 1 convention: 0 = success,
 *     negative = argument / system error, positive = the operation ran but access was refused.
 *   - IV is exactly 96 bits, tag exactly 128 bits (reading S5).
 *   - len <= 2^36 - 32 bytes (SP 800-38D), aad_len < 2^61 bytes.  len = 0 and / or aad_len = 0 are
 *     valid and the matching pointers may then be NULL (reading S6).
 *   - In place (out == in) is allowed; any other overlap of in and out is GCM_ERR_ARG.
 *   - Any byte alignment is accepted; the fast path needs `in` and `out` 16-byte aligned.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the default stream).
 *   - A gcm_ctx may be used by one call at a time (it owns the cross-CTA scratch of that call): a call that
 *     finds the context in use by another thread returns GCM_ERR_BUSY and does nothing.  Asynchronous calls
 *     on one context must be issued to one stream (or otherwise ordered) so that their kernels do not overlap.
 *   - Every call runs on the context's device and leaves the calling thread's current CUDA device as it was.
 *   - On GCM_ERR_AUTH the whole output [0, len) has been overwritten with zeros (the paper's payload
 *     suppression) and the call completes normally (L245).  The fused kernel writes
 *     plaintext before the tag is known (reading S9); the synchronous call does not return before
 *     the compare and, on failure, the wipe have completed.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns
 *     GCM_ERR_CUDA.
 */
#ifndef B200_GCM_H
#define B200_GCM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define GCM_API __attribute__((visibility("default")))
#else
#define GCM_API
#endif

typedef struct gcm_ctx gcm_ctx; /* opaque */

enum {
    GCM_OK        = 0,
    GCM_ERR_AUTH  = 1,   /* tag mismatch: plaintext output has been zero-filled                 */
    GCM_ERR_ARG   = -1,  /* NULL pointer, key_bits not 128/256, partial overlap, bad geometry    */
    GCM_ERR_LEN   = -2,  /* len > 2^36 - 32 bytes, or aad_len >= 2^61 bytes                      */
    GCM_ERR_CUDA  = -3,  /* CUDA runtime failure; see gcm_last_cuda_error()                      */
    GCM_ERR_NOMEM = -4,
    GCM_ERR_BUSY  = -5   /* the context is in use by another call                                */
};

/* Library / build identification: "b200gcm <version> sm_100a". Never NULL. */
GCM_API const char *gcm_version(void);

/* Selects the CUDA device (ordinal) on which subsequent gcm_init / batch / gfc_context_create calls of the
 * process make their contexts; -1 (the default) = the calling thread's current CUDA device at the time of the
 * call.  Does not change the caller's current device.  A context stays on the device it was made on.
 * Returns GCM_OK, GCM_ERR_ARG (no such device) or GCM_ERR_CUDA. */
GCM_API int gcm_set_device(int ordinal);

/* Last cudaError_t seen by the library (0 = none), and its text (host, static storage). */
GCM_API int gcm_last_cuda_error(void);
GCM_API const char *gcm_last_cuda_error_string(void);

/*
 * gcm_init -- step a1 + a2 of SURVEY.md 8(a): key schedule (FIPS-197 5.2), H = E_K(0^128), the
 * powers of H the reduction uses ("table of powers of the hash key",
 * generated on the GPU) and the multiplier table of the fixed stride power.  Runs one setup
 * kernel on the selected device.
 *   out      (host, out)  receives the new context
 *   key      (host)       16 or 32 bytes
 *   key_bits              128 or 256 (reading S1); anything else -> GCM_ERR_ARG
 */
GCM_API int gcm_init(gcm_ctx **out, const uint8_t *key, int key_bits);

/* Zeroises key material (device tables, host copy of the round keys) and frees the context.
 * NULL is ignored. */
GCM_API void gcm_destroy(gcm_ctx *ctx);

/*
 * Launch geometry of the fused kernel: at most `grid` CTAs (0 = one per SM) of `threads` threads (256, 384
 * or 512; 0 = default 512).  No table depends on it (the GHASH stride power is H^32 for every launch shape), and
 * results never depend on the geometry (geometry-agnostic counters; reading S11).
 * Under the default geometry, messages of at most 511 GHASH blocks (AAD blocks + payload blocks + the length
 * block, about 8 KiB) take a single-CTA latency kernel instead; an explicit geometry always selects the
 * fused kernel.  Returns GCM_OK / GCM_ERR_ARG / GCM_ERR_CUDA.
 */
GCM_API int gcm_set_geometry(gcm_ctx *ctx, int grid, int threads);
GCM_API int gcm_get_geometry(const gcm_ctx *ctx, int *grid, int *threads);

/*
 * Which unit does the GF(2^128) multiplies of GHASH (step a7 of the path; Eq. 1 leaves the method
 * of the multiply open, reading S7):
 *   GCM_GHASH_TABLE   an 8-bit Shoup table of the stride power K = H^32 in shared memory, 16 reads of 16 bytes per
 *                     block (gcm_fused.cu), for every call;
 *   GCM_GHASH_TENSOR  the tensor cores: the multiply as a GF(2) matrix-vector product, tcgen05.mma kind::mxf4 with
 *                     0 / 1 operands, accumulators in TMEM, parity of the counts.  Encrypt / decrypt of at least 8 MiB
 *                     with 16-byte aligned buffers run gcm_tc2.cu (AES warps and tensor-core GHASH warps side by side)
 *                     between two short launches of the row kernel (AAD and first blocks; rest and length block);
 *                     shorter or unaligned messages run gcm_tc.cu (the row kernel with a7 on the tensor cores);
 *                     gcm_ghash_async on at least 4 MiB of aligned input runs gcm_ghash_tc.cu.  `threads` of
 *                     gcm_set_geometry is ignored by these kernels, `grid` kept;
 *   GCM_GHASH_AUTO    (default) what is fastest on a B200: the tensor-core kernels for aligned messages of at least
 *                     384 MiB (AES-128: 128 MiB) and for gcm_ghash_async on at least 32 MiB, the table otherwise.
 * Results are bit-identical under all three.  The batched calls and the latency kernel are not affected.
 * Returns GCM_OK / GCM_ERR_ARG.
 */
enum { GCM_GHASH_TABLE = 0, GCM_GHASH_TENSOR = 1, GCM_GHASH_AUTO = 2 };
GCM_API int gcm_set_ghash_engine(gcm_ctx *ctx, int engine);
GCM_API int gcm_get_ghash_engine(const gcm_ctx *ctx, int *engine);

/*
 * Diagnostics for the roofline (the pipe bound must use MEASURED unit rates): runs
 * a short probe on the current device and writes thread-operations per SM-cycle, averaged over the
 * SMs, for the instruction classes the kernels are made of.  rates (host, out) has room for n >=
 * GCM_RATE_COUNT doubles, indexed by the enum below.  Returns GCM_OK / GCM_ERR_ARG / GCM_ERR_CUDA.
 * Not part of the data path.
 */
enum {
    GCM_RATE_LDS32 = 0,     /* conflict-free 4-byte shared-memory reads (the AES table read)        */
    GCM_RATE_LDS128,        /* conflict-free 16-byte shared-memory reads (the GHASH table read)     */
    GCM_RATE_LOP3,          /* three-input logic                                                     */
    GCM_RATE_PRMT,          /* byte permute (table address formation)                                */
    GCM_RATE_IMAD,          /* 32-bit integer multiply-add                                           */
    GCM_RATE_IMAD_WIDE,     /* 32 x 32 + 64 -> 64 multiply-add (the generic GF(2^128) product)       */
    GCM_RATE_LOP3_IMAD,     /* LOP3 and IMAD interleaved 1:1 (both pipes), operations of both kinds  */
    GCM_RATE_MMA_MXF4,      /* tensor pipe: 128 x 128 x 64 tcgen05.mma kind::mxf4 back to back, in GHASH blocks
                               (128 x 128 bit products) per SM-cycle, not thread-operations                 */
    GCM_RATE_COUNT
};
GCM_API int gcm_measure_pipe_rates(double *rates, int n);

/*
 * Diagnostics: per-phase time stamps of the fused kernel.  d_stamps (device) has room for
 * 8 x uint64 per CTA of the largest grid used (GCM_PHASE_SLOTS x grid x 8 bytes); while it is set, thread 0 of
 * every CTA stores %globaltimer (ns) at: [0] kernel entry, [1] tables in shared memory, [2] after
 * griddepcontrol.wait, [3] its rows done, [4] all warps' partials in, [5] ticket drawn, [6] finisher done (last CTA
 * only), [7] position weights formed by warp 0 (between [1] and [2]).  NULL switches it off (the default).  Not part
 * of the data path.
 */
#define GCM_PHASE_SLOTS 8
GCM_API int gcm_set_phase_stamps(gcm_ctx *ctx, void *d_stamps);

/*
 * Diagnostics for the host logic (no CUDA call, usable without a GPU): the launch layout the library derives from
 * the lengths of a message, and the chunk plan of the host-buffer pipeline.  Tests check their invariants and model
 * the kernels' GHASH regrouping on the CPU from them.
 *   gcm_debug_row_layout: virtual block sequence [pad | AAD | payload | length block] of one launch;
 *     ctr_base = index of the launch's first payload block within its message, last = the launch ends the message,
 *     aligned = the buffers are 16-byte aligned.  Returns GCM_OK / GCM_ERR_ARG / GCM_ERR_LEN.
 *   gcm_debug_plan_chunks: chunk lengths of gcm_encrypt_host for a message of `len` bytes into plan[0 .. cap);
 *     returns the number of chunks, or GCM_ERR_ARG when cap is too small.
 */
typedef struct {
    uint64_t vblocks;        /* E: pad + AAD blocks + payload blocks + length block                         */
    uint64_t base;           /* virtual index of payload block 0                                            */
    uint32_t pad;            /* leading zero blocks, 0..31                                                   */
    uint32_t n_aad_blocks;
    uint32_t rows;           /* ceil(E / 32)                                                                 */
    uint32_t fast_lo, fast_hi; /* rows [fast_lo, fast_hi) hold only whole payload blocks                     */
    uint32_t ctr_delta;      /* counter of virtual block v = (uint32)v + ctr_delta                           */
    uint32_t len_block;      /* 1: the last virtual block is the length block                                */
    uint32_t reserved;
} gcm_row_layout;
GCM_API int gcm_debug_row_layout(uint64_t len, uint64_t aad_len, uint32_t ctr_base, int last, int aligned, gcm_row_layout *out);
GCM_API int gcm_debug_plan_chunks(uint64_t len, uint64_t *plan, uint32_t cap);

/*
 * Diagnostics: the SM clock the tensor-core kernel of the long-message path (gcm_tc2_kernel) ran at in
 * this context's most recent call, measured by the kernel itself: CTA 0 stores clock64() and %globaltimer at its entry
 * and exit into the context's scratch (four words, always, not a data-path branch).  nvidia-smi keeps reporting the
 * maximum clock while a tcgen05 kernel runs several per cent below it, so the roofline of bench.py uses this value.
 *   sm_mhz     host, out: SM cycles per microsecond over CTA 0's lifetime
 *   kernel_ms  host, out: that lifetime in milliseconds
 * Synchronises the device.  Returns GCM_OK, GCM_ERR_ARG (NULL argument, or no such kernel has run on the context),
 * GCM_ERR_BUSY or GCM_ERR_CUDA.
 */
GCM_API int gcm_debug_tc2_clock(gcm_ctx *ctx, double *sm_mhz, double *kernel_ms);

/* Copies the hash subkey H = E_K(0^128) (16 bytes) to host memory; for tests of step a2. */
GCM_API int gcm_get_hash_subkey(const gcm_ctx *ctx, uint8_t h[16]);

/*
 * gcm_encrypt -- SURVEY.md 8(a) steps a3-a11, SP 800-38D Algorithm 4 (GCM-AE_K(IV, P, A)):
 *   C = P xor E_K(IV || BE32(g + 2)) per 16-byte block g (counter from the block index only,
 *   PAPER.md L259-L270); T = E_K(IV || 0^31 || 1) xor GHASH_H(A || 0* || C || 0* || len64(A) || len64(C)).
 *   iv    (host)    12 bytes
 *   d_aad (device)  aad_len bytes, may be NULL when aad_len = 0
 *   d_pt  (device)  len bytes, may be NULL when len = 0
 *   d_ct  (device)  len bytes, out
 *   tag   (host)    16 bytes, out
 * Synchronises `cuda_stream` before returning.
 */
GCM_API int gcm_encrypt(gcm_ctx *ctx, const uint8_t iv[12],
                const void *d_aad, uint64_t aad_len,
                const void *d_pt, uint64_t len,
                void *d_ct, uint8_t tag[16], void *cuda_stream);

/*
 * gcm_decrypt_verify -- SP 800-38D Algorithm 5 (GCM-AD) with the paper's validation gate
 * and payload suppression (L243): recomputes the tag from (IV, A, C), compares
 * it with `tag` in constant time on the device, and returns GCM_OK with P in d_pt, or
 * GCM_ERR_AUTH with d_pt[0..len) all zero.
 *   tag   (host)    16 bytes, in
 * Synchronises `cuda_stream` before returning.
 */
GCM_API int gcm_decrypt_verify(gcm_ctx *ctx, const uint8_t iv[12],
                       const void *d_aad, uint64_t aad_len,
                       const void *d_ct, uint64_t len,
                       void *d_pt, const uint8_t tag[16], void *cuda_stream);

/*
 * Asynchronous forms for device-timed measurement (the paper's protocol places cudaEvent pairs
 * strictly around the kernels): same computation, tag / status stay on the device,
 * no synchronisation, no host transfer.
 *   d_tag    (device) 16 bytes: out for encrypt, in (expected tag) for decrypt
 *   d_status (device) one int32: GCM_OK or GCM_ERR_AUTH; on GCM_ERR_AUTH d_pt is zero-filled by a
 *            wipe kernel enqueued on the same stream.
 */
GCM_API int gcm_encrypt_async(gcm_ctx *ctx, const uint8_t iv[12],
                      const void *d_aad, uint64_t aad_len,
                      const void *d_pt, uint64_t len,
                      void *d_ct, void *d_tag, void *cuda_stream);

GCM_API int gcm_decrypt_verify_async(gcm_ctx *ctx, const uint8_t iv[12],
                             const void *d_aad, uint64_t aad_len,
                             const void *d_ct, uint64_t len,
                             void *d_pt, const void *d_tag, void *d_status, void *cuda_stream);

/*
 * Host-buffer forms (the paper's data plane stages files through pinned host memory and overlaps
 * the transfers with the kernels on CUDA streams): `h_*` are HOST
 * pointers (pinned memory gives full PCIe rate; pageable memory works).  The message is cut into
 * chunks (2 MiB at both ends of the message, doubling to at most 64 MiB in the middle) that travel H2D -> fused kernel -> D2H on three internal
 * streams; the running GHASH state is handed from chunk to chunk on the device.  The plaintext of chunk k is copied
 * out before the tag of the whole message is known (reading S9); gcm_decrypt_verify_host_strict does not do that.  Work already queued on `cuda_stream`
 * is waited for; the call returns when the output and the tag / verdict are in host memory.
 * On GCM_ERR_AUTH h_pt[0..len) is zero-filled.  aad_len < 2^32 here.
 */
GCM_API int gcm_encrypt_host(gcm_ctx *ctx, const uint8_t iv[12],
                     const void *h_aad, uint64_t aad_len,
                     const void *h_pt, uint64_t len,
                     void *h_ct, uint8_t tag[16], void *cuda_stream);

GCM_API int gcm_decrypt_verify_host(gcm_ctx *ctx, const uint8_t iv[12],
                            const void *h_aad, uint64_t aad_len,
                            const void *h_ct, uint64_t len,
                            void *h_pt, const uint8_t tag[16], void *cuda_stream);

/*
 * Strict form of gcm_decrypt_verify_host: verify-then-release at the API level.  Pass 1
 * streams the ciphertext through the GHASH-only kernel (no AES on the payload, nothing written to h_pt) and
 * compares the tag on the device; only if it matches does pass 2 decrypt into h_pt.  No byte of unverified
 * plaintext ever reaches the caller's buffer (on GCM_ERR_AUTH h_pt is left untouched), at the price of a second
 * host-to-device transfer of the ciphertext.
 */
GCM_API int gcm_decrypt_verify_host_strict(gcm_ctx *ctx, const uint8_t iv[12],
                                   const void *h_aad, uint64_t aad_len,
                                   const void *h_ct, uint64_t len,
                                   void *h_pt, const uint8_t tag[16], void *cuda_stream);

/*
 * GHASH only (GMAC-style measurement; the paper's Table 5 "GHashKernelOnly",
 * PAPER.md L363, L379-L392): S = GHASH_H(A || 0* || C || 0* || len64(A) || len64(C)) over
 * device-resident data, 16 bytes written to d_out (device).  No AES on the payload.
 */
GCM_API int gcm_ghash_async(gcm_ctx *ctx, const void *d_aad, uint64_t aad_len,
                    const void *d_c, uint64_t len, void *d_out, void *cuda_stream);

/*
 * Batched many-message variant (FITS-sized HDUs and many short messages).
 * One descriptor per message; keys may differ per message.
 *   key      (host)   16 or 32 bytes       key_bits 128 or 256
 *   iv                12 bytes
 *   d_aad    (device) aad_len bytes        d_in / d_out (device) len bytes
 *   tag               out (encrypt) / in (decrypt)
 *   status            per message: GCM_OK / GCM_ERR_AUTH / negative error
 * gcm_encrypt_batch returns GCM_OK or the first negative error.
 * gcm_decrypt_verify_batch returns the number of messages that failed authentication (their
 * outputs are zero-filled) or a negative error.  Both synchronise `cuda_stream`.
 */
typedef struct {
    const uint8_t *key;
    int            key_bits;
    uint8_t        iv[12];
    const void    *d_aad;
    uint64_t       aad_len;
    const void    *d_in;
    uint64_t       len;
    void          *d_out;
    uint8_t        tag[16];
    int            status;
} gcm_msg;

GCM_API int gcm_encrypt_batch(gcm_msg *msgs, uint32_t n, void *cuda_stream);
GCM_API int gcm_decrypt_verify_batch(gcm_msg *msgs, uint32_t n, void *cuda_stream);

/*
 * Device-descriptor form of the batched calls, for many short messages (config C4): the descriptors
 * themselves live in DEVICE memory, so a call marshals nothing on the host (for 10,000 messages that is a quarter of
 * the synchronous call's time) and does not synchronise: one small kernel orders the messages longest first, one
 * persistent warp-per-message kernel per key size does the work, and every message's tag (encrypt) and verdict are
 * written into its own descriptor.  The caller fills the array once (keys included: it is the caller's to wipe) and
 * may launch it any number of times.
 *   key       16 or 32 bytes used          key_bits  128 or 256 (anything else: status = GCM_ERR_ARG, message skipped)
 *   tag       out (encrypt) / in (decrypt) status    out: GCM_OK / GCM_ERR_AUTH (output zero-filled) / GCM_ERR_ARG / GCM_ERR_LEN
 *   iv        12 bytes                     d_aad / d_in / d_out (device), aad_len, len as in gcm_msg
 * Every message is handled by one warp whatever its length: meant for messages up to a few hundred KiB (longer ones
 * are correct but slow; use gcm_encrypt_batch for FITS-sized messages).  The ordering kernel checks what it can see
 * of each descriptor: len > 2^36 - 32 or aad_len >= 2^36 gives status GCM_ERR_LEN, a NULL d_in / d_out / d_aad with
 * a non-zero length GCM_ERR_ARG, and such messages are skipped like one with a bad key_bits.  Overlap rules are the
 * caller's to keep (the descriptors cannot be checked from the host).  Calls on different streams are ordered behind
 * each other by the library.  Returns GCM_OK or a negative error for the launch itself.
 */
typedef struct {
    uint8_t     key[32];
    uint8_t     tag[16];
    int32_t     status;
    uint32_t    key_bits;
    uint8_t     iv[12];
    uint32_t    reserved;
    const void *d_aad;
    const void *d_in;
    void       *d_out;
    uint64_t    aad_len;
    uint64_t    len;
} gcm_dmsg;                     /* 112 bytes */

GCM_API int gcm_encrypt_batch_device(gcm_dmsg *d_msgs, uint32_t n, void *cuda_stream);
GCM_API int gcm_decrypt_verify_batch_device(gcm_dmsg *d_msgs, uint32_t n, void *cuda_stream);

/* Frees the batch path's cached per-key contexts and staging buffers (zeroising key material) and the
 * wiped allocations that gcm_destroy keeps for the next gcm_init. */
GCM_API void gcm_batch_release(void);

#ifdef __cplusplus
}
#endif

#endif /* B200_GCM_H */
