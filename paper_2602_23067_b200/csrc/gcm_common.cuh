// gcm_common.cuh -- constants, table layouts and launch-parameter structs shared by the kernels
// and the host side of libb200gcm.so.  Shares nothing with oracle/.
#pragma once
#include <stdint.h>

// ---- shared-memory layout of the fused kernel (bytes) -------------------------------------------
// AES round tables, laid out so that every lane of a warp owns one 4-byte bank (conflict-free AND
// constant-time for secret indices).  Row x (x = S-box input, 0..255) is 256 bytes:
//     A0: [T0[x] for lanes 0..31][T1[x] for lanes 0..31]      A1: [T2[x] ..][T3[x] ..]
// so the byte address of T_k[x] for a lane is  x*256 + lane*4 (+128 for the odd table): one PRMT
// builds it from the state byte and the lane offset, no shift / multiply needed.
#define AES_A0_OFF      0
#define AES_A1_OFF      65536
#define AES_ODD_OFF     128
#define AES_TAB_BYTES   131072
// GHASH multiplier table for the fixed stride power K = H^32 (a warp's 32 lanes hold 32 consecutive
// blocks, so every lane's next block is 32 blocks further on): 8-bit Shoup tables, one per byte
// position P = 0..15.  Entry (P, v) = (block with byte P = v, zero elsewhere) . K, 16 bytes in memory
// byte order, stored at  v*256 + (P>>3)*128 + (P&7)*16.  Within a quarter-warp lane q visits
// positions in the rotated order (q + r) & 7, so the eight 16-byte accesses of one LDS.128 phase fall
// into eight distinct bank groups: conflict-free without replication.
#define KTAB_OFF        131072
#define KTAB_BYTES      65536
#define RED_OFF         (KTAB_OFF + KTAB_BYTES)     /* cross-warp reduction scratch: 32 x 16 B */
#define RED_BYTES       512
#define WPOW_OFF        (RED_OFF + RED_BYTES)       /* per-warp position weights D_w: 32 x 16 B */
#define WPOW_BYTES      512
#define MBAR_OFF        (WPOW_OFF + WPOW_BYTES)     /* one mbarrier (8 B) for the bulk copy of ktab */
#define FUSED_SMEM_BYTES (MBAR_OFF + 16)

// ---- GHASH on the tensor cores (gcm_tc.cu) ------------------------------------------------------
// A lane's TC_L consecutive blocks and its running value make one chunk = TC_L + 1 slices of one tcgen05.mma tile;
// slice weights are K^0 .. K^TC_L (K = H^32), one 8 KB bit matrix each (the MMA's B operand, in shared memory).
#define TC_L              8
#define TC_BMAT_BYTES     8192
#define TC_BMAT_TOTAL     ((TC_L + 1) * TC_BMAT_BYTES)
#define TC_PRODUCER_WARPS 12          /* + one warp that issues the MMAs: 416 threads per CTA */

// GHASH-only on the tensor cores (gcm_ghash_tc.cu): chunks of GT_L slices of 128 consecutive blocks; slice weights are
// powers of H^128, the chunk-to-chunk multiplier H^(128 GT_L) goes through an 8-bit table.
#define GT_L              16
#define GT_CHUNK_BLOCKS   (128 * GT_L)
#define GT_BMAT_TOTAL     (GT_L * TC_BMAT_BYTES)
#define GT_MIN_BYTES      (4ull << 20)   /* GCM_GHASH_TENSOR: shorter messages stay with the row kernels */
#define GT_AUTO_BYTES     (32ull << 20)  /* GCM_GHASH_AUTO: its prologue (192 KB of tables, TMEM) costs the tensor kernel about 3 us
                                            more than the table kernel; it is level at 32 MiB and ahead beyond */

// AES-CTR + tensor-core GHASH with separate warps (gcm_tc2.cu): the stretch starts at payload block T2_HEAD_BLOCKS, whose
// counter (block index + 2) is 0 mod 256, and is a whole number of 128-block slices.
#define T2_HEAD_BLOCKS    254
#define T2_MIN_BYTES      (8ull << 20)      /* GCM_GHASH_TENSOR: from here on gcm_tc2.cu, below it gcm_tc.cu */
#define T2_AUTO_BYTES_256 (384ull << 20)    /* GCM_GHASH_AUTO: a chain costs 25-30 us more than it would at its steady rate; level with */
#define T2_AUTO_BYTES_128 (128ull << 20)    /* the table kernel at 230 MiB (AES-256) / 96 MiB (AES-128), ahead beyond */

#define GCM_MAX_THREADS 512
#define GCM_MAX_GRID    4096
#define GCM_MAX_DEVICES 64
#define GCM_STRIDE      32          /* blocks between a lane's consecutive blocks: K = H^GCM_STRIDE */

// Powers of H for position weights (PAPER.md L197 precomputes H^(2^k); four radix-512 digits need
// two tree levels instead of up to 36):  hx[k*512 + j] = H^(j * 512^k), k = 0..3, j = 0..511.
#define HX_DIGITS       4
#define HX_RADIX_BITS   9
#define HX_ENTRIES      (HX_DIGITS << HX_RADIX_BITS)
#define GCM_MAX_VBLOCKS (1ull << (HX_DIGITS * HX_RADIX_BITS))   /* virtual GHASH blocks per launch */

enum { MODE_ENCRYPT = 0, MODE_DECRYPT = 1, MODE_GHASH = 2 };

// Device-resident per-key tables (owned by gcm_ctx).
struct GcmTables {
    const uint32_t *te0;     // 256 words: T0[x] = {02.S, S, S, 03.S} (little-endian word, row 0 low); host copy: gcm_ctx::h_te0
    const uint4    *ktab;    // KTAB_BYTES, layout above
    const uint4    *hpow;    // hpow[i] = H^i, i = 0..GCM_STRIDE ("mem" format)
    const uint4    *hx;      // HX_ENTRIES radix-512 powers
    const uint4    *h;       // H
    const uint4    *bmat;    // TC_BMAT_TOTAL: bit matrices of K^0 .. K^TC_L for the tensor-core GHASH (gcm_tc.cu)
};

// One message as the row loop (gcm_device.cuh: gcm_rows) sees it.
//
// Virtual block sequence:  [pad zero blocks][AAD blocks][payload blocks][length block], E blocks in all, cut
// into rows of 32.  A warp owns a contiguous stretch of rows, so a lane's consecutive blocks are always 32
// apart (one fixed GHASH multiplier K = H^32 for every geometry) and their counters differ only in the low
// byte for 8 rows at a time (rounds 1-2 are mostly cached).  pad (0..31) is chosen so that
// counter = virtual index + ctr_delta with ctr_delta = 0 mod 32; leading zero blocks are free in GHASH.
// The length block BE64(8 aad) || BE64(8 len) (a10) is the last virtual block of the launch that finishes a
// message (len_block = 1): it is hashed like any other block, so the tag needs no product after the combine.
struct RowMsg {
    const uint8_t *in;
    uint8_t       *out;
    const uint8_t *aad;
    uint64_t len;            // payload bytes of this launch
    uint64_t aad_len;
    uint64_t base;           // pad + n_aad_blocks: virtual index of payload block 0
    uint64_t vblocks;        // E: pad + AAD blocks + payload blocks + len_block
    uint64_t final_len;      // whole-message lengths for the length block
    uint64_t final_aad_len;
    uint32_t pad;            // leading virtual zero blocks
    uint32_t n_aad_blocks;
    uint32_t rows;           // S = ceil(E / 32)
    uint32_t fast_lo, fast_hi; // rows [fast_lo, fast_hi) hold only whole payload blocks of aligned buffers
    uint32_t aligned;        // in and out are 16-byte aligned
    uint32_t ctr_delta;      // counter of the block at virtual index v is (uint32)v + ctr_delta
    uint32_t len_block;      // 1: the last virtual block is the length block
};

// Host-side (and device-side, for the warp-per-message kernel) derivation of a RowMsg from lengths and pointers.
// ctr_base: index of the first payload block of this launch within its message (0 except in the chunked host
// pipeline).  len_block: this launch finishes the message.
__host__ __device__ __forceinline__ void row_msg_fill(RowMsg &d, const uint8_t *in, uint8_t *out, const uint8_t *aad,
                                                      uint64_t len, uint64_t aad_len, uint32_t ctr_base, uint32_t len_block,
                                                      uint64_t final_len, uint64_t final_aad_len, bool ghash_only)
{
    const uint64_t n_full = len / 16, n_blocks = (len + 15) / 16, n_aad = (aad_len + 15) / 16;
    d.in = in; d.out = out; d.aad = aad;
    d.len = len; d.aad_len = aad_len;
    d.final_len = final_len; d.final_aad_len = final_aad_len;
    // leading zero blocks (free in GHASH) make counter == virtual index (mod 32)
    d.pad = (2u + ctr_base - (uint32_t)n_aad) & (GCM_STRIDE - 1);
    d.n_aad_blocks = (uint32_t)n_aad;
    d.base = (uint64_t)d.pad + n_aad;
    d.len_block = len_block;
    d.vblocks = d.base + n_blocks + len_block;
    d.rows = (uint32_t)((d.vblocks + GCM_STRIDE - 1) / GCM_STRIDE);
    d.ctr_delta = ctr_base + 2u - (uint32_t)d.base;
    const uintptr_t a = (uintptr_t)in, b = ghash_only ? 0 : (uintptr_t)out;
    d.aligned = ((a | b) & 15) == 0 ? 1u : 0u;
    d.fast_lo = d.fast_hi = 0;
    if (d.aligned) {
        d.fast_lo = (uint32_t)((d.base + GCM_STRIDE - 1) / GCM_STRIDE);
        d.fast_hi = (uint32_t)((d.base + n_full) / GCM_STRIDE);
        if (d.fast_hi < d.fast_lo) d.fast_hi = d.fast_lo;
    }
}

// Kernel parameters of the single-message kernels, passed by value (constant bank): the round keys are then
// free operands of the XOR instructions.  Warp w (global index) of W owns rows [w*S/W, (w+1)*S/W).
struct GcmParams {
    uint32_t rk[60];         // round keys, little-endian column words: rk[4r + c]
    uint32_t te0[256];       // the round table T0 (key-independent): expanded into shared memory at kernel start
    uint32_t iv[3];          // IV words (little-endian load of bytes 0..11)
    uint32_t warps;          // W: warps the rows are dealt to (grid * warps per CTA)
    RowMsg   m;
    GcmTables tab;
    uint4    *partials;      // one per CTA
    unsigned *counter;       // last-CTA-done ticket: counts up for the life of the context, never reset
    unsigned  ticket_last;   // the ticket that makes a CTA of THIS launch the finisher (epoch scheme)
    uint32_t  status_init;   // 1: CTA 0 stores GCM_STATUS_PENDING into *status first (device-resident verdict words)
    uint4    *tag_out;       // device, 16 bytes (encrypt: tag; ghash mode: S)
    const uint4 *tag_in;     // device, 16 bytes or NULL -> tag_expect below
    uint32_t tag_expect[4];
    int      *status;        // device (or mapped host): GCM_STATUS_PENDING at kernel start, then 0 / 1
    // chunked (host-pipeline) operation: this launch covers payload blocks [ctr_base, ...) of a longer
    // message.  chain_in/chain_pow: running GHASH state before this chunk and H^(GHASH blocks of this
    // chunk); chain_out != NULL: store the new running state instead of finishing the tag.
    const uint4 *chain_in;
    const uint4 *chain_pow;
    uint4    *chain_out;
    unsigned long long *stamps;   // diagnostics (gcm_set_phase_stamps): 8 x u64 of %globaltimer per CTA, or NULL
};

// Verdict word before the finisher has written it: anything but 0 is a refusal (fail closed).
#define GCM_STATUS_PENDING 0x7FFFFFFF
