// gcm_tc.cuh -- host entry points of the fused kernel with GHASH on the tensor cores (gcm_tc.cu).
#pragma once
#include <cuda_runtime.h>
#include "gcm_common.cuh"

// nr: 10 or 14; mode: MODE_*; blocks: CTAs to launch.  p.warps must be blocks * TC_PRODUCER_WARPS.
cudaError_t launch_tc(int nr, int mode, int blocks, const GcmParams &p, cudaStream_t s);
// bmat[e] = bit matrix of "multiply by H^(32 e)", e = 0 .. TC_L, from the context's power table hx (once per key)
void launch_tc_setup(const uint4 *hx, uint4 *bmat, cudaStream_t s);
