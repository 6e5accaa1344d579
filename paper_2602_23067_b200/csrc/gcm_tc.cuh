// gcm_tc.cuh -- host entry points of the fused kernel with GHASH on the tensor cores (gcm_tc.cu).
#pragma once
#include <cuda_runtime.h>
#include "gcm_common.cuh"

// nr: 10 or 14; mode: MODE_*; blocks: CTAs to launch.  p.warps must be blocks * TC_PRODUCER_WARPS.
cudaError_t launch_tc(int nr, int mode, int blocks, const GcmParams &p, cudaStream_t s);
// bmat[e] = bit matrix of "multiply by H^(32 e)", e = 0 .. TC_L, from the context's power table hx (once per key)
void launch_tc_setup(const uint4 *hx, uint4 *bmat, cudaStream_t s);

// gcm_ghash_tc.cu: GHASH_H(A, C) of a 16-byte-aligned C in ONE launch on the tensor cores: the virtual sequence
// [pad | AAD | C | length block] in whole chunks of GT_CHUNK_BLOCKS.  Tables: launch_ghash_tc_setup, once per key.
static inline uint64_t ghash_tc_chunks(uint64_t aad_len, uint64_t len)
{
    return ((aad_len + 15) / 16 + (len + 15) / 16 + 1 + GT_CHUNK_BLOCKS - 1) / GT_CHUNK_BLOCKS;
}
void launch_ghash_tc_setup(const uint4 *hx, uint4 *bmat2, uint4 *ktab2, cudaStream_t s);
cudaError_t launch_ghash_tc(int blocks, const uint8_t *aad, uint64_t aad_len, const uint8_t *in, uint64_t len, const uint4 *bmat2,
                            const uint4 *ktab2, const uint4 *hx, uint4 *partials, unsigned *counter, unsigned ticket_last, uint4 *out,
                            cudaStream_t s);

// gcm_tc2.cu: AES-CTR + GHASH of nslices * 128 whole aligned blocks (AES warps apart from the tensor-core GHASH), one
// link of a chunk chain.
cudaError_t launch_tc2(int nr, int mode, int blocks, const uint32_t *rk, const uint32_t *te0, const uint8_t *iv, uint32_t ctr0,
                       const uint8_t *in, uint8_t *out, uint64_t nslices, const uint4 *bmat2, const uint4 *hx, uint4 *partials,
                       unsigned *counter, unsigned ticket_last, const uint4 *chain_in, uint4 *chain_out, uint64_t exp_next,
                       uint4 *pow_out, unsigned long long *clk, cudaStream_t s);
