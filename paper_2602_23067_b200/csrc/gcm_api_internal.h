// gcm_api_internal.h -- the context behind the opaque gcm_ctx of include/gcm.h (host side only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>
#include <atomic>

// memset that the compiler may not drop as a dead store (parameter blocks hold round keys, staging holds raw keys;
// runs at memory speed, not byte by byte)
static inline void secure_zero(void *p, size_t n)
{
    memset(p, 0, n);
    __asm__ __volatile__("" : : "r"(p) : "memory");
}

struct HostPipe;          // gcm_host.cu: staging buffers, streams and events of the host-buffer entry points

struct gcm_ctx {
    int device;
    int key_bits;
    int nr;            // 10 / 14
    int sm_count;
    int grid;          // CTAs of the fused kernel at most (default: one per SM)
    int threads;       // threads per CTA (512 default, 256 / 384 alternatives)
    int engine;        // GCM_GHASH_TABLE / _TENSOR / _AUTO (gcm_set_ghash_engine)
    // device state, one slab
    uint8_t  *d_slab;
    size_t    slab_bytes;
    uint32_t *d_te0;
    uint32_t *d_rk;
    uint4    *d_h;
    uint4    *d_hpow;
    uint4    *d_hx;
    uint4    *d_ktab;
    uint4    *d_bmat;     // bit matrices of K^0 .. K^TC_L (gcm_tc.cu)
    uint4    *d_bmat2;    // bit matrices of H^(128 e), e < GT_L, and the multiplier table of H^(128 GT_L) (gcm_ghash_tc.cu)
    uint4    *d_ktab2;
    uint4    *d_gt;       // chain scratch of the three-launch tensor path (gcm_tc2.cu): state behind the head, behind the stretch, chain power of the tail
    uint4    *d_partials;
    unsigned *d_counter;
    uint4    *d_tag;
    int      *d_status;
    unsigned long long *d_stamps;   // gcm_set_phase_stamps: caller-owned diagnostics buffer or NULL
    // host state
    // host copies for the kernel parameter block, in the slab's order so that one copy fetches both
    uint32_t  h_te0[256]; // round table T0
    uint32_t  h_rk[64];   // round keys (little-endian column words), 60 used
    uint8_t  *h_pinned;   // 64 bytes of mapped pinned memory: tag [0,16), status [16,20)
    unsigned  ticket_next;  // tickets handed to launches so far (the device counter is never reset)
    std::atomic<int> busy;  // 1 while a call owns the context (its cross-CTA scratch, pinned block, pipeline)
    HostPipe *pipe;       // lazily created by gcm_encrypt_host / gcm_decrypt_verify_host
};

// One call at a time per context: the second caller gets GCM_ERR_BUSY instead of racing on the scratch.
struct CtxLock {
    gcm_ctx *c;
    bool ok;
    explicit CtxLock(gcm_ctx *ctx) : c(ctx), ok(false)
    {
        int expect = 0;
        if (c) ok = c->busy.compare_exchange_strong(expect, 1, std::memory_order_acquire);
    }
    ~CtxLock() { if (ok) c->busy.store(0, std::memory_order_release); }
    CtxLock(const CtxLock &) = delete;
    CtxLock &operator=(const CtxLock &) = delete;
};

// Makes `device` current for the scope of a call and restores the caller's device afterwards.
struct DeviceGuard {
    int prev;
    cudaError_t err;
    explicit DeviceGuard(int device) : prev(-1), err(cudaSuccess)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
        else if (err != cudaSuccess) prev = -1;
    }
    ~DeviceGuard()
    {
        int now = -1;
        if (prev >= 0 && cudaGetDevice(&now) == cudaSuccess && now != prev) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

int gcm_cuda_fail(cudaError_t e);
// The device new contexts are made on: the one chosen by gcm_set_device, else the calling thread's current device.
int gcm_default_device(int *device);
// gcm_init on an explicit device (the batch and container layers pass the device their staging lives on)
int gcm_init_on_device(gcm_ctx **out, const uint8_t *key, int key_bits, int device);
int gcm_sm_count(int device, int *sms);
struct GcmParams;
// Argument checks and launch parameters common to encrypt / decrypt / ghash.  ctr_base: index of the first payload
// block of this launch within its message; last: this launch finishes the message (appends the length block).
// Hands the launch its finishing ticket: call exactly once per launch that is then actually made.
int gcm_build_params(gcm_ctx *c, int mode, const uint8_t *iv, const void *d_aad, uint64_t aad_len,
                     const void *d_in, uint64_t len, void *d_out, uint32_t ctr_base, bool last,
                     uint64_t final_len, uint64_t final_aad_len, GcmParams *p, int *blocks);
// launch_fused with the context's geometry; gives the tickets back if the launch could not be made
cudaError_t gcm_launch_fused(gcm_ctx *c, int mode, int blocks, const GcmParams &p, cudaStream_t s);
void gcm_host_pipe_free(gcm_ctx *c);
// gcm_host.cu: the chunked host-buffer pipeline behind gcm_encrypt_host / gcm_decrypt_verify_host (the caller
// holds the context lock).  mode MODE_GHASH: h_out unused, tag_io receives GHASH_H(A, C).
int gcm_host_run(gcm_ctx *c, int mode, const uint8_t *iv, const void *h_aad, uint64_t aad_len,
                 const void *h_in, uint64_t len, void *h_out, uint8_t *tag_io, void *user_stream,
                 unsigned long long *d_sum32);
// gcm_api.cu: frees the pooled (wiped) allocations of destroyed contexts.
void gcm_pool_release(void);
