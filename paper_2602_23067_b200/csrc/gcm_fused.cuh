// gcm_fused.cuh -- host entry point of the fused CTR + GHASH kernel.
#pragma once
#include <cuda_runtime.h>
#include "gcm_common.cuh"

// nr: 10 or 14; mode: MODE_*; threads: 256 or 512; blocks: CTAs to launch
cudaError_t launch_fused(int nr, int mode, int threads, int blocks, const GcmParams &p, cudaStream_t s);
