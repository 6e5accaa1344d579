// gcm_setup.cuh -- launch parameters and host entry points of the setup / wipe kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct SetupParams {
    uint32_t key[8];     // raw key bytes as little-endian words (by value: never staged in global memory)
    int      key_bits;   // 128 or 256
    int      threads;    // threads per CTA of the fused kernel
    int      grid;       // CTAs of the fused kernel
    uint32_t *te0;       // out: 256 words
    uint32_t *rk;        // out: 60 words, little-endian column words
    uint4    *h;         // out (setup) / in (regeometry): H
    uint4    *hpow;      // out: threads + 1 entries
    uint4    *bpow;      // out: grid + 1 entries
    uint4    *ktab;      // out: 4096 entries
};

__device__ void gcm_build_power_tables(uint4 h, int threads, int grid, uint4 *hpow, uint4 *bpow, uint4 *ktab, uint4 *s_v);

void launch_setup(const SetupParams &p, cudaStream_t s);
void launch_regeometry(const SetupParams &p, cudaStream_t s);
void launch_wipe(uint8_t *dst, uint64_t len, const int *status, cudaStream_t s);
