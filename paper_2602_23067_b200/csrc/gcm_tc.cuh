// gcm_tc.cuh -- host entry points of the fused kernel with GHASH on the tensor cores (gcm_tc.cu).
#pragma once
#include <cuda_runtime.h>
#include "gcm_common.cuh"

// nr: 10 or 14; mode: MODE_*; blocks: CTAs to launch.  p.warps must be blocks * TC_PRODUCER_WARPS.
cudaError_t launch_tc(int nr, int mode, int blocks, const GcmParams &p, cudaStream_t s);
// bmat[e] = bit matrix of "multiply by H^(32 e)", e = 0 .. TC_L, from the context's power table hx (once per key)
void launch_tc_setup(const uint4 *hx, uint4 *bmat, cudaStream_t s);

// gcm_ghash_tc.cu: GHASH of nchunks * GT_CHUNK_BLOCKS aligned blocks as one link of a chunk chain (chain_in may be
// NULL); also stores H^exp_next to pow_out for the launch that follows.  Tables: launch_ghash_tc_setup, once per key.
void launch_ghash_tc_setup(const uint4 *hx, uint4 *bmat2, uint4 *ktab2, cudaStream_t s);
cudaError_t launch_ghash_tc(int blocks, const uint8_t *in, uint64_t nchunks, const uint4 *bmat2, const uint4 *ktab2, const uint4 *hx,
                            uint4 *partials, unsigned *counter, unsigned ticket_last, const uint4 *chain_in, uint4 *chain_out,
                            uint64_t exp_next, uint4 *pow_out, cudaStream_t s);
