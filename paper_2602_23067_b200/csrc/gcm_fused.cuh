// gcm_fused.cuh -- host entry point of the fused CTR + GHASH kernel.
#pragma once
#include <cuda_runtime.h>
#include "gcm_common.cuh"

// nr: 10 or 14; mode: MODE_*; threads: 256 or 512; blocks: CTAs to launch
cudaError_t launch_fused(int nr, int mode, int threads, int blocks, const GcmParams &p, cudaStream_t s);

// gcm_small.cu: single-CTA latency kernel for messages of at most SMALL_MAX_BLOCKS GHASH blocks
// (AAD blocks + payload blocks + the length block, if any); MODE_ENCRYPT / MODE_DECRYPT only; chain_in / chain_pow /
// chain_out of a chunk chain are honoured (the links of gcm_tc2.cu).
#define SMALL_MAX_BLOCKS 511
cudaError_t launch_small(int nr, int mode, const GcmParams &p, cudaStream_t s);

// gcm_fused.cu: shared launch helpers.  launch_with_pdl launches with programmatic stream serialization (the
// kernel must call griddepcontrol.wait before it touches stream-ordered data); ensure_smem_attr raises the
// dynamic shared-memory limit of `kern` once per device (configured: GCM_MAX_DEVICES flags owned by the caller).
#include <atomic>
cudaError_t launch_with_pdl(const void *kern, dim3 grid, dim3 block, size_t smem, cudaStream_t s, void **args);
cudaError_t ensure_smem_attr(const void *kern, std::atomic<bool> *configured, size_t bytes);
