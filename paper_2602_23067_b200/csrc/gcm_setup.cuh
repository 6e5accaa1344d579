// gcm_setup.cuh -- launch parameters and host entry points of the setup / wipe kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct SetupParams {
    uint32_t key[8];     // raw key bytes as little-endian words (by value: never staged in global memory)
    int      key_bits;   // 128 or 256
    uint32_t *te0;       // out: 256 words
    uint32_t *rk;        // out: 60 words, little-endian column words
    uint4    *h;         // out: H
    uint4    *hpow;      // out: GCM_STRIDE + 1 entries
    uint4    *hx;        // out: HX_ENTRIES entries
    uint4    *ktab;      // out: 4096 entries
};

__device__ void gcm_build_power_tables(uint4 h, uint4 *hpow, uint4 *hx, uint4 *ktab, uint4 *s_v);

void launch_setup(const SetupParams &p, cudaStream_t s);
void launch_te0(uint32_t *te0, cudaStream_t s);
void launch_wipe(uint8_t *dst, uint64_t len, const int *status, cudaStream_t s);
