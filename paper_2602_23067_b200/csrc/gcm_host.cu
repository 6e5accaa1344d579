// gcm_host.cu -- host-buffer entry points (gcm_encrypt_host / gcm_decrypt_verify_host).
//
// The paper's data plane stages files through pinned host memory and overlaps transfers with the
// kernels on CUDA streams (section 3.3.2, L288-L293 section 5.2.3).  Here the
// message is cut into chunks; chunk k travels  H2D -> fused kernel -> D2H  on stream k mod 3, so the
// copy engines run both directions while the SMs work on another chunk.  The kernels are serialised
// among themselves by events because each one hands the running GHASH state to the next:
//     Y_k = Y_(k-1) . H^(n_k)  xor  Horner(chunk k)          (n_k = GHASH blocks of chunk k)
// which is Eq. 1 regrouped; H^(n_k) comes from a small power kernel that runs
// while the first chunk is still on the wire.
#include <cuda_runtime.h>
#include <string.h>
#include <new>

#include "../../include/gcm.h"
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_setup.cuh"
#include "gcm_fused.cuh"
#include "gcm_api_internal.h"
#include "fits_sum.cuh"

#ifndef PIPE_SLOTS
#define PIPE_SLOTS 3
#endif
#ifndef PIPE_CHUNK_BYTES
#define PIPE_CHUNK_BYTES (64ull << 20)   /* staging buffer = largest chunk; multiple of PIPE_MIN_CHUNK_BYTES */
#endif
#ifndef PIPE_MIN_CHUNK_BYTES
#define PIPE_MIN_CHUNK_BYTES (2ull << 20)   /* first and last chunk: what the pipeline cannot overlap */
#endif
#ifndef PIPE_ZEROCOPY_MAX_BYTES
#define PIPE_ZEROCOPY_MAX_BYTES (4ull << 20)   /* up to here a pinned message is read and written in place over PCIe */
#endif
#define PIPE_MAX_CHUNKS ((uint32_t)((1ull << 36) / PIPE_CHUNK_BYTES) + 76)   /* 2^36 bytes in full chunks + the two ramps */

struct HostPipe {
    cudaStream_t stream[PIPE_SLOTS];
    cudaEvent_t kernel_done[PIPE_SLOTS];
    cudaEvent_t start;
    uint8_t *d_stage[PIPE_SLOTS];
    uint8_t *d_aad;
    size_t aad_cap;
    uint4 *d_state;     // [2]: running GHASH state, ping-pong
    uint4 *d_pows;      // [PIPE_MAX_CHUNKS]: H^(GHASH blocks of chunk k)
    uint64_t *d_exp;    // [PIPE_MAX_CHUNKS]: those block counts
    uint64_t *h_exp;    // pinned staging of d_exp
};

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) return gcm_cuda_fail(e__);                                         \
    } while (0)

// out[k] = H^(e[k]), e[k] < 2^36, one thread per exponent: the product of four entries of the context's radix-512
// digit tables hx[d*512 + j] = H^(j * 512^d) ("table of powers of the hash key").
__global__ void gcm_chunk_pow_kernel(const uint4 *hx, const uint64_t *e, uint32_t n, uint4 *out)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const uint64_t d = e[k];
    const uint32_t mask = (1u << HX_RADIX_BITS) - 1;
    gf128 r = gf_from_mem(hx[(uint32_t)d & mask]);
    for (uint32_t dig = 1; dig < HX_DIGITS; dig++) {
        const uint32_t j = (uint32_t)(d >> (HX_RADIX_BITS * dig)) & mask;
        if (j) r = gf_mul(r, gf_from_mem(hx[(dig << HX_RADIX_BITS) + j]));
    }
    out[k] = gf_to_mem(r);
}

// Chunk lengths of a message of `len` bytes.  Measured on the B200 box (per-chunk event timeline, 64 MiB message):
// with both directions busy every copy costs about 30 us on top of its bytes at 50 GB/s (a 4 MiB copy takes 113 us,
// not 84), so the plan wants FEW chunks, while the first upload and the last download, which overlap with nothing,
// want SMALL ones.  Hence: PIPE_MIN_CHUNK_BYTES at both ends, doubling up to the middle size (about len / 4, at most
// PIPE_CHUNK_BYTES) and coming down again by a factor of about 0.6 per chunk (a chunk's slot is wanted again three
// chunks later, so the sizes must not fall faster than the downloads drain).  Every chunk but the last is a multiple
// of PIPE_MIN_CHUNK_BYTES (so of 16); the last one takes the ragged end.
static uint32_t plan_chunks(uint64_t len, uint64_t *plan)
{
    if (len == 0) { plan[0] = 0; return 1; }
    const uint64_t U = PIPE_MIN_CHUNK_BYTES;
    uint64_t mid = U;
    while (mid * 2 <= len / 4 && mid * 2 <= PIPE_CHUNK_BYTES) mid *= 2;
    uint64_t back[PIPE_MAX_CHUNKS];
    uint32_t nf = 0, nb = 0;
    const uint64_t last = ((len - 1) % U) + 1;
    uint64_t rem = len - last;
    back[nb++] = last;
    uint64_t a = U, b = (U * 8 / 5 + U - 1) / U * U;
    if (b > mid) b = mid;
    while (rem > 0) {
        uint64_t t = a < rem ? a : rem;
        plan[nf++] = t; rem -= t;
        a = a * 2 < mid ? a * 2 : mid;
        if (rem > 0) {
            t = b < rem ? b : rem;
            back[nb++] = t; rem -= t;
            b = (b * 8 / 5 + U - 1) / U * U;            // x 1.6, rounded up to the unit
            if (b > mid) b = mid;
        }
    }
    for (uint32_t i = nb; i-- > 0;) plan[nf++] = back[i];
    return nf;
}

static void pipe_destroy(HostPipe *hp)
{
    if (!hp) return;
    for (int i = 0; i < PIPE_SLOTS; i++) {
        if (hp->stream[i]) cudaStreamSynchronize(hp->stream[i]);
        if (hp->d_stage[i]) {
            launch_wipe(hp->d_stage[i], PIPE_CHUNK_BYTES, nullptr, 0);
            cudaDeviceSynchronize();
            cudaFree(hp->d_stage[i]);
        }
        if (hp->kernel_done[i]) cudaEventDestroy(hp->kernel_done[i]);
        if (hp->stream[i]) cudaStreamDestroy(hp->stream[i]);
    }
    if (hp->start) cudaEventDestroy(hp->start);
    if (hp->d_aad) cudaFree(hp->d_aad);
    if (hp->d_state) cudaFree(hp->d_state);
    if (hp->d_exp) cudaFree(hp->d_exp);
    if (hp->h_exp) cudaFreeHost(hp->h_exp);
    cudaGetLastError();
    delete hp;
}

// The pipeline is built in a local and attached to the context only when complete: a failed allocation (192 MiB
// of staging) leaves the context as it was, and the next call tries again.
static int pipe_get(gcm_ctx *c, size_t aad_len)
{
    if (!c->pipe) {
        HostPipe *hp = new (std::nothrow) HostPipe;
        if (!hp) return GCM_ERR_NOMEM;
        memset(hp, 0, sizeof(*hp));
        cudaError_t e = cudaSuccess;
        for (int i = 0; i < PIPE_SLOTS && e == cudaSuccess; i++) {
            if ((e = cudaStreamCreateWithFlags(&hp->stream[i], cudaStreamNonBlocking)) != cudaSuccess) break;
            if ((e = cudaEventCreateWithFlags(&hp->kernel_done[i], cudaEventDisableTiming)) != cudaSuccess) break;
            e = cudaMalloc((void **)&hp->d_stage[i], PIPE_CHUNK_BYTES);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hp->start, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaMalloc((void **)&hp->d_state, (2 + PIPE_MAX_CHUNKS) * sizeof(uint4));
        if (e == cudaSuccess) e = cudaMalloc((void **)&hp->d_exp, PIPE_MAX_CHUNKS * sizeof(uint64_t));
        if (e == cudaSuccess) e = cudaHostAlloc((void **)&hp->h_exp, PIPE_MAX_CHUNKS * sizeof(uint64_t), cudaHostAllocDefault);
        if (e != cudaSuccess) {
            pipe_destroy(hp);
            return gcm_cuda_fail(e);
        }
        hp->d_pows = hp->d_state + 2;
        c->pipe = hp;
    }
    HostPipe *hp = c->pipe;
    if (aad_len > hp->aad_cap) {
        if (hp->d_aad) cudaFree(hp->d_aad);
        hp->d_aad = nullptr;
        hp->aad_cap = 0;
        size_t cap = (aad_len + 4095) & ~(size_t)4095;
        CU(cudaMalloc((void **)&hp->d_aad, cap));
        hp->aad_cap = cap;
    }
    return GCM_OK;
}

void gcm_host_pipe_free(gcm_ctx *c)
{
    pipe_destroy(c->pipe);
    c->pipe = nullptr;
}

// d_sum32 (device, may be NULL): every chunk's ciphertext is also added to the FITS DATASUM accumulator
// while it is still in the staging buffer (the container layer of gfc_frame.cu).
// mode MODE_GHASH: the chunks are only hashed (no AES, nothing copied back): tag_io receives GHASH_H(A, C).
int gcm_host_run(gcm_ctx *c, int mode, const uint8_t *iv, const void *h_aad, uint64_t aad_len,
                 const void *h_in, uint64_t len, void *h_out, uint8_t *tag_io, void *user_stream,
                 unsigned long long *d_sum32)
{
    if (!c || (!iv && mode != MODE_GHASH) || !tag_io) return GCM_ERR_ARG;
    if (len > ((1ull << 36) - 32) || aad_len >= (1ull << 32)) return GCM_ERR_LEN;
    if ((aad_len && !h_aad) || (len && (!h_in || (!h_out && mode != MODE_GHASH)))) return GCM_ERR_ARG;
    int rc = pipe_get(c, aad_len);
    if (rc != GCM_OK) return rc;
    HostPipe *hp = c->pipe;
    cudaStream_t us = (cudaStream_t)user_stream;
    // An error return after the first enqueue must not leave copies in flight on the caller's h_in / h_out: every
    // early return below drains the pipeline streams first (the success paths have synchronised already).
    struct Drain {
        HostPipe *hp;
        bool armed;
        ~Drain() { if (armed) for (int i = 0; i < PIPE_SLOTS; i++) cudaStreamSynchronize(hp->stream[i]); }
    } drain{hp, true};

    // Short messages in pinned (or registered) host memory skip the staging copies altogether: under unified
    // addressing the kernel reads the plaintext and writes the ciphertext in place over PCIe, one launch, no DMA
    // set-up (measured on the B200 box: 1 MiB 57 us against 81 us staged; equal at 16 MiB; beyond that the copy
    // engines win: kernel loads and stores together reach 30 GB/s, the two copy engines 2 x 50).
    if (len > 0 && len <= PIPE_ZEROCOPY_MAX_BYTES && mode != MODE_GHASH && d_sum32 == nullptr) {
        cudaPointerAttributes ai, ao;
        if (cudaPointerGetAttributes(&ai, h_in) == cudaSuccess && cudaPointerGetAttributes(&ao, h_out) == cudaSuccess &&
            ai.type == cudaMemoryTypeHost && ao.type == cudaMemoryTypeHost && ai.devicePointer && ao.devicePointer) {
            cudaStream_t s0 = hp->stream[0];
            CU(cudaEventRecord(hp->start, us));
            CU(cudaStreamWaitEvent(s0, hp->start, 0));
            if (aad_len) CU(cudaMemcpyAsync(hp->d_aad, h_aad, aad_len, cudaMemcpyHostToDevice, s0));
            GcmParams p;
            int blocks = 0;
            rc = gcm_build_params(c, mode, iv, aad_len ? hp->d_aad : nullptr, aad_len, ai.devicePointer, len, ao.devicePointer,
                                  0, true, len, aad_len, &p, &blocks);
            if (rc != GCM_OK) return rc;
            if (mode == MODE_DECRYPT) memcpy(p.tag_expect, tag_io, 16);
            volatile int *verdict0 = (volatile int *)(c->h_pinned + 16);
            *verdict0 = GCM_STATUS_PENDING;
            p.tag_out = (uint4 *)c->h_pinned;
            p.status = (int *)(c->h_pinned + 16);
            cudaError_t e = gcm_launch_fused(c, mode, blocks, p, s0);
            secure_zero(&p, sizeof(p));
            if (e != cudaSuccess) return gcm_cuda_fail(e);
            CU(cudaStreamSynchronize(s0));
            drain.armed = false;
            if (mode == MODE_ENCRYPT) { memcpy(tag_io, c->h_pinned, 16); return GCM_OK; }
            if (*verdict0 != 0) { memset(h_out, 0, len); return GCM_ERR_AUTH; }
            return GCM_OK;
        }
        cudaGetLastError();          // pageable memory: cudaPointerGetAttributes may leave an error behind on old drivers
    }

    // chunk plan: small chunks at both ends, PIPE_CHUNK_BYTES in the middle
    uint64_t plan[PIPE_MAX_CHUNKS];
    const uint32_t n_chunks = plan_chunks(len, plan);
    // work already queued on the caller's stream happens before ours
    CU(cudaEventRecord(hp->start, us));
    for (int i = 0; i < PIPE_SLOTS; i++) CU(cudaStreamWaitEvent(hp->stream[i], hp->start, 0));
    if (aad_len) CU(cudaMemcpyAsync(hp->d_aad, h_aad, aad_len, cudaMemcpyHostToDevice, hp->stream[0]));
    if (n_chunks > 1) {
        // chain_pow of chunk k: H^(GHASH blocks of chunk k) = its payload blocks, plus the length block in the last
        cudaStream_t sp = hp->stream[PIPE_SLOTS - 1];
        for (uint32_t k = 0; k < n_chunks; k++) hp->h_exp[k] = (plan[k] + 15) / 16 + (k == n_chunks - 1 ? 1 : 0);
        CU(cudaMemcpyAsync(hp->d_exp, hp->h_exp, n_chunks * sizeof(uint64_t), cudaMemcpyHostToDevice, sp));
        gcm_chunk_pow_kernel<<<(n_chunks + 63) / 64, 64, 0, sp>>>(c->d_hx, hp->d_exp, n_chunks, hp->d_pows);
        CU(cudaGetLastError());
        CU(cudaEventRecord(hp->kernel_done[PIPE_SLOTS - 1], sp));
    }
    // the verdict reads "refused" until the finisher of the last chunk has written it (fail closed)
    volatile int *verdict = (volatile int *)(c->h_pinned + 16);
    *verdict = GCM_STATUS_PENDING;

    uint64_t off = 0;
    for (uint32_t k = 0; k < n_chunks; off += plan[k], k++) {
        const int slot = (int)(k % PIPE_SLOTS);
        cudaStream_t s = hp->stream[slot];
        const uint64_t clen = plan[k];
        const bool first = (k == 0), last = (k == n_chunks - 1);
        if (clen) CU(cudaMemcpyAsync(hp->d_stage[slot], (const uint8_t *)h_in + off, clen, cudaMemcpyHostToDevice, s));
        // kernels run in message order: chunk k needs chunk k-1's GHASH state (and the powers)
        if (!first) CU(cudaStreamWaitEvent(s, hp->kernel_done[(k - 1) % PIPE_SLOTS], 0));
        else if (n_chunks > 1) CU(cudaStreamWaitEvent(s, hp->kernel_done[PIPE_SLOTS - 1], 0));

        GcmParams p;
        int blocks = 0;
        rc = gcm_build_params(c, mode, iv, first ? hp->d_aad : nullptr, first ? aad_len : 0,
                              hp->d_stage[slot], clen, mode == MODE_GHASH ? nullptr : hp->d_stage[slot],
                              (uint32_t)(off / 16), last, len, aad_len, &p, &blocks);
        if (rc != GCM_OK) return rc;
        if (!first) {
            p.chain_in = hp->d_state + ((k - 1) & 1);
            p.chain_pow = hp->d_pows + k;
        }
        if (!last) p.chain_out = hp->d_state + (k & 1);
        if (mode == MODE_DECRYPT) memcpy(p.tag_expect, tag_io, 16);
        // tag / verdict of the last chunk go straight into mapped pinned host memory
        p.tag_out = (uint4 *)c->h_pinned;
        p.status = (int *)(c->h_pinned + 16);
        cudaError_t e = gcm_launch_fused(c, mode, blocks, p, s);
        secure_zero(&p, sizeof(p));
        if (e != cudaSuccess) return gcm_cuda_fail(e);
        CU(cudaEventRecord(hp->kernel_done[slot], s));
        if (d_sum32 && mode == MODE_ENCRYPT) CU(launch_fits_sum32(hp->d_stage[slot], clen, d_sum32, c->sm_count, s));
        if (clen && mode != MODE_GHASH) CU(cudaMemcpyAsync((uint8_t *)h_out + off, hp->d_stage[slot], clen, cudaMemcpyDeviceToHost, s));
    }
    for (int i = 0; i < PIPE_SLOTS; i++) CU(cudaStreamSynchronize(hp->stream[i]));
    drain.armed = false;
    if (mode != MODE_DECRYPT) {
        memcpy(tag_io, c->h_pinned, 16);
        return GCM_OK;
    }
    if (*verdict != 0) {
        memset(h_out, 0, len);       // payload suppression on the host copy
        return GCM_ERR_AUTH;
    }
    return GCM_OK;
}

#define LOCK_CTX(c)                                                                                \
    if (!(c)) return GCM_ERR_ARG;                                                                  \
    CtxLock lock__(c);                                                                             \
    if (!lock__.ok) return GCM_ERR_BUSY;                                                           \
    DeviceGuard guard__((c)->device);                                                              \
    CU(guard__.err)

extern "C" int gcm_debug_plan_chunks(uint64_t len, uint64_t *plan, uint32_t cap)
{
    if (!plan || len > ((1ull << 36) - 32)) return GCM_ERR_ARG;
    uint64_t full[PIPE_MAX_CHUNKS];
    const uint32_t n = plan_chunks(len, full);
    if (n > cap) return GCM_ERR_ARG;
    memcpy(plan, full, n * sizeof(uint64_t));
    return (int)n;
}

extern "C" int gcm_encrypt_host(gcm_ctx *c, const uint8_t iv[12], const void *h_aad, uint64_t aad_len,
                                const void *h_pt, uint64_t len, void *h_ct, uint8_t tag[16], void *stream)
{
    LOCK_CTX(c);
    return gcm_host_run(c, MODE_ENCRYPT, iv, h_aad, aad_len, h_pt, len, h_ct, tag, stream, nullptr);
}

extern "C" int gcm_decrypt_verify_host(gcm_ctx *c, const uint8_t iv[12], const void *h_aad, uint64_t aad_len,
                                       const void *h_ct, uint64_t len, void *h_pt, const uint8_t tag[16], void *stream)
{
    if (!tag) return GCM_ERR_ARG;
    LOCK_CTX(c);
    uint8_t t[16];
    memcpy(t, tag, 16);
    return gcm_host_run(c, MODE_DECRYPT, iv, h_aad, aad_len, h_ct, len, h_pt, t, stream, nullptr);
}

// E_K(J0) xor S compared with the expected tag on the device (constant time), verdict into mapped pinned memory.
__global__ void gcm_tag_check_kernel(const uint4 *ekj0, const uint4 *s, uint4 expect, int *status)
{
    const uint4 t = xor4(*ekj0, *s);
    const uint32_t diff = (t.x ^ expect.x) | (t.y ^ expect.y) | (t.z ^ expect.z) | (t.w ^ expect.w);
    *status = diff != 0 ? 1 : 0;
}

extern "C" int gcm_decrypt_verify_host_strict(gcm_ctx *c, const uint8_t iv[12], const void *h_aad, uint64_t aad_len,
                                              const void *h_ct, uint64_t len, void *h_pt, const uint8_t tag[16], void *stream)
{
    if (!tag || !iv) return GCM_ERR_ARG;
    LOCK_CTX(c);
    // pass 1: S = GHASH_H(A, C) over the host buffer (H2D + GHASH-only kernel per chunk, no AES, no output)
    uint8_t s_host[16];
    int rc = gcm_host_run(c, MODE_GHASH, nullptr, h_aad, aad_len, h_ct, len, nullptr, s_host, stream, nullptr);
    if (rc != GCM_OK) return rc;
    // E_K(J0) = tag of the empty message with empty AAD (S = 0) through the latency kernel; compare on the device
    HostPipe *hp = c->pipe;
    cudaStream_t s = hp->stream[0];
    {
        GcmParams p;
        int blocks = 0;
        rc = gcm_build_params(c, MODE_ENCRYPT, iv, nullptr, 0, nullptr, 0, nullptr, 0, true, 0, 0, &p, &blocks);
        if (rc != GCM_OK) return rc;
        c->ticket_next -= (unsigned)blocks;                      // the latency kernel draws no tickets
        p.tag_out = hp->d_state;                                 // E_K(J0)
        cudaError_t e = launch_small(c->nr, MODE_ENCRYPT, p, s);
        secure_zero(&p, sizeof(p));
        if (e != cudaSuccess) return gcm_cuda_fail(e);
    }
    CU(cudaMemcpyAsync(hp->d_state + 1, s_host, 16, cudaMemcpyHostToDevice, s));
    volatile int *verdict = (volatile int *)(c->h_pinned + 16);
    *verdict = GCM_STATUS_PENDING;
    uint4 expect;
    memcpy(&expect, tag, 16);
    gcm_tag_check_kernel<<<1, 1, 0, s>>>(hp->d_state, hp->d_state + 1, expect, (int *)(c->h_pinned + 16));
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(s));
    if (*verdict != 0) return GCM_ERR_AUTH;                      // nothing was written to h_pt
    // pass 2: the ordinary pipeline (which verifies once more while it decrypts)
    uint8_t t[16];
    memcpy(t, tag, 16);
    return gcm_host_run(c, MODE_DECRYPT, iv, h_aad, aad_len, h_ct, len, h_pt, t, stream, nullptr);
}
