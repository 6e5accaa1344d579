// gcm_api_internal.h -- the context behind the opaque gcm_ctx of include/gcm.h (host side only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct HostPipe;          // gcm_host.cu: staging buffers, streams and events of the host-buffer entry points

struct gcm_ctx {
    int device;
    int key_bits;
    int nr;            // 10 / 14
    int sm_count;
    int grid;          // CTAs of the fused kernel at most (default: one per SM)
    int threads;       // threads per CTA (512 default, 256 alternative)
    // device state, one slab
    uint8_t  *d_slab;
    size_t    slab_bytes;
    uint32_t *d_te0;
    uint32_t *d_rk;
    uint4    *d_h;
    uint4    *d_hpow;
    uint4    *d_hx;
    uint4    *d_ktab;
    uint4    *d_partials;
    unsigned *d_counter;
    uint4    *d_tag;
    int      *d_status;
    // host state
    uint32_t  h_rk[60];   // round keys (little-endian column words) for the kernel parameter block
    uint8_t  *h_pinned;   // 64 bytes of pinned memory: tag [0,16), status [16,20)
    HostPipe *pipe;       // lazily created by gcm_encrypt_host / gcm_decrypt_verify_host
};

int gcm_cuda_fail(cudaError_t e);
struct GcmParams;
int gcm_build_params(gcm_ctx *c, int mode, const uint8_t *iv, const void *d_aad, uint64_t aad_len,
                     const void *d_in, uint64_t len, void *d_out, uint32_t ctr_base, GcmParams *p, int *blocks);
void gcm_host_pipe_free(gcm_ctx *c);
// gcm_host.cu: the chunked host-buffer pipeline behind gcm_encrypt_host / gcm_decrypt_verify_host.
int gcm_host_run(gcm_ctx *c, int mode, const uint8_t *iv, const void *h_aad, uint64_t aad_len,
                 const void *h_in, uint64_t len, void *h_out, uint8_t *tag_io, void *user_stream,
                 unsigned long long *d_sum32);
// gcm_api.cu: frees the pooled (wiped) allocations of destroyed contexts.
void gcm_pool_release(void);
