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
#define FUSED_SMEM_BYTES (RED_OFF + RED_BYTES)

#define GCM_MAX_THREADS 512
#define GCM_MAX_GRID    4096
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
    const uint32_t *te0;     // 256 words: T0[x] = {02.S, S, S, 03.S} (little-endian word, row 0 low)
    const uint4    *ktab;    // KTAB_BYTES, layout above
    const uint4    *hpow;    // hpow[i] = H^i, i = 0..GCM_STRIDE ("mem" format)
    const uint4    *hx;      // HX_ENTRIES radix-512 powers
    const uint4    *h;       // H
};

// Kernel parameters, passed by value (constant bank): the round keys are then free operands of
// the XOR instructions.
//
// Virtual block sequence of one launch:  [pad zero blocks][AAD blocks][payload blocks], E blocks in
// all, cut into rows of 32.  Warp w (global index) owns rows [w*Q, (w+1)*Q): a contiguous stretch, so
// a lane's consecutive blocks are always 32 apart (one fixed GHASH multiplier for every geometry)
// and their counters differ only in the low byte for 8 rows at a time (rounds 1-2 are mostly cached).
// pad (0..31) is chosen so that counter = virtual index + ctr_delta with ctr_delta = 0 mod 32.
struct GcmParams {
    uint32_t rk[60];         // round keys, little-endian column words: rk[4r + c]
    uint32_t iv[3];          // IV words (little-endian load of bytes 0..11)
    const uint8_t *in;
    uint8_t       *out;
    const uint8_t *aad;
    uint64_t len;            // payload bytes
    uint64_t aad_len;
    uint64_t base;           // pad + n_aad_blocks: virtual index of payload block 0
    uint64_t vblocks;        // E: pad + AAD blocks + payload blocks
    uint32_t pad;            // leading virtual zero blocks
    uint32_t n_aad_blocks;
    uint32_t rows;           // S = ceil(E / 32)
    uint32_t rows_per_warp;  // Q
    uint32_t fast_lo, fast_hi; // rows [fast_lo, fast_hi) hold only whole payload blocks of aligned buffers
    uint32_t aligned;        // in and out are 16-byte aligned
    uint32_t ctr_delta;      // counter of the block at virtual index v is (uint32)v + ctr_delta
    GcmTables tab;
    uint4    *partials;      // one per CTA
    unsigned *counter;       // last-CTA-done ticket
    uint4    *tag_out;       // device, 16 bytes (encrypt: tag; ghash mode: S)
    const uint4 *tag_in;     // device, 16 bytes or NULL -> tag_expect below
    uint32_t tag_expect[4];
    int      *status;        // device
    // chunked (host-pipeline) operation: this launch covers payload blocks [ctr_base, ...) of a longer
    // message.  chain_in/chain_pow: running GHASH state before this chunk and H^(GHASH blocks of this
    // chunk); chain_out != NULL: store the new running state instead of finishing the tag.
    const uint4 *chain_in;
    const uint4 *chain_pow;
    uint4    *chain_out;
    uint64_t final_len;      // whole-message lengths for the length block
    uint64_t final_aad_len;
};
