// gcm_rates.cu -- gcm_measure_pipe_rates(): the unit rates the roofline of DESIGN.md section 6 is built
// from, measured on the device the library runs on ("measure it, do not assume").
// One 512-thread CTA per SM, eight independent dependency chains per thread, clock64 per SM; the
// result is thread-operations per SM-cycle, averaged over the SMs.  Diagnostics only: nothing on the
// data path depends on it.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gcm.h"
#include "gcm_api_internal.h"

#define RATE_ITERS  1024
#define RATE_CHAINS 8
#define RATE_THREADS 512

template <int OP>
__global__ void __launch_bounds__(RATE_THREADS, 1)
gcm_rate_kernel(uint32_t *sink, long long *cycles, uint32_t seed)
{
    __shared__ __align__(16) uint32_t sm[8192];
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) sm[i] = (i * 4) & 0x7FF0;   // valid byte offsets
    __syncthreads();
    uint32_t r[RATE_CHAINS];
    uint64_t w[RATE_CHAINS];
    const uint32_t lane4 = (threadIdx.x & 31) * 4;
#pragma unroll
    for (int c = 0; c < RATE_CHAINS; c++) { r[c] = seed + threadIdx.x * 7 + c; w[c] = r[c]; }
    const uint32_t k1 = seed | 1, k2 = seed * 3 + 5;
    const uint32_t saddr = (uint32_t)__cvta_generic_to_shared(sm);
    const long long t0 = clock64();
#pragma unroll 4
    for (int it = 0; it < RATE_ITERS; it++) {
#pragma unroll
        for (int c = 0; c < RATE_CHAINS; c++) {
            if (OP == GCM_RATE_LDS32)      // every lane its own bank, data-dependent row: the AES table read
                asm volatile("{ .reg .u32 a; and.b32 a, %0, 0x7F80; add.u32 a, a, %1; ld.shared.u32 %0, [a]; }"
                             : "+r"(r[c]) : "r"(saddr + lane4));
            if (OP == GCM_RATE_LDS128) {   // 16 bytes per lane, conflict-free: the GHASH table read
                uint32_t a1, a2, a3;
                asm volatile("{ .reg .u32 a; and.b32 a, %0, 0x7E00; add.u32 a, a, %4; ld.shared.v4.u32 {%0, %1, %2, %3}, [a]; }"
                             : "+r"(r[c]), "=r"(a1), "=r"(a2), "=r"(a3) : "r"(saddr + lane4 * 4));
                r[c] ^= (a1 ^ a2 ^ a3) & 1;
            }
            if (OP == GCM_RATE_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[c]) : "r"(k1), "r"(k2));
            if (OP == GCM_RATE_PRMT) asm volatile("prmt.b32 %0, %0, %1, 0x5140;" : "+r"(r[c]) : "r"(k1));
            if (OP == GCM_RATE_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[c]) : "r"(k1), "r"(k2));
            if (OP == GCM_RATE_IMAD_WIDE) asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(w[c]) : "r"(r[c]), "r"(k1));
            if (OP == GCM_RATE_LOP3_IMAD) {
                if (c & 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[c]) : "r"(k1), "r"(k2));
                else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[c]) : "r"(k1), "r"(k2));
            }
        }
    }
    const long long t1 = clock64();
    uint32_t acc = 0;
#pragma unroll
    for (int c = 0; c < RATE_CHAINS; c++) acc ^= r[c] ^ (uint32_t)w[c] ^ (uint32_t)(w[c] >> 32);
    sink[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// The tensor pipe as gcm_tc.cu / gcm_ghash_tc.cu use it: 128 x 128 x 64 tcgen05.mma kind::mxf4 (e2m1 operands, A from
// TMEM, B from shared memory, fp32 accumulators in TMEM, all scale factors 2^0), issued back to back by one elected
// lane into two alternating accumulators.  One such MMA multiplies 64 bits of 128 GHASH blocks by a 64 x 128 bit
// slice of a matrix, i.e. it is worth 64 blocks: the rate reported is GHASH blocks per SM-cycle.
#define RATE_MMAS 2048
__global__ void __launch_bounds__(128, 1)
gcm_rate_mma_kernel(long long *cycles)
{
    extern __shared__ __align__(1024) uint8_t sm[];          // [0, 4096): a B tile (no-swizzle K-major), then an mbarrier and the TMEM base
    uint64_t *bar = reinterpret_cast<uint64_t *>(sm + 4096);
    uint32_t *tslot = reinterpret_cast<uint32_t *>(sm + 4096 + 16);
    const uint32_t t = threadIdx.x, warp = t >> 5;
    for (uint32_t i = t; i < 1024; i += 128) reinterpret_cast<uint32_t *>(sm)[i] = 0x22222222u;       // 1.0 everywhere
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    const uint32_t bar_a = (uint32_t)__cvta_generic_to_shared(bar);
    if (t == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((uint32_t)__cvta_generic_to_shared(tslot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tb = __shfl_sync(0xFFFFFFFFu, *tslot, 0), lanebase = tb + ((32u * warp) << 16);
    {
        const uint32_t one = 0x7F7F7F7Fu, x = 0x11111111u;    // scale factors 2^0 at columns [256, 288); A = 0.5 everywhere at [288, 296)
        for (int c = 0; c < 32; c += 8)
            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(lanebase + 256 + c), "r"(one) : "memory");
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(lanebase + 288), "r"(x) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (warp == 0) {
        const uint32_t saddr = (uint32_t)__cvta_generic_to_shared(sm);
        const uint64_t desc = (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(2048 >> 4) << 16) | ((uint64_t)(128 >> 4) << 32) | (1ull << 46);
        const uint32_t idesc = (1u << 7) | (1u << 10) | (16u << 17) | (1u << 23) | (8u << 24);
        uint32_t pred;
        asm volatile("{ .reg .pred p; elect.sync _|p, 0xFFFFFFFF; selp.u32 %0, 1, 0, p; }" : "=r"(pred));
        if (pred) {
            const long long t0 = clock64();
#pragma unroll 4
            for (int i = 0; i < RATE_MMAS; i++)
                asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %5, 0;\n"
                             "tcgen05.mma.cta_group::1.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%4], [%4], p;\n}"
                             ::"r"(tb + 128 * (i & 1)), "r"(tb + 288), "l"(desc), "r"(idesc), "r"(tb + 256), "r"(i > 1 ? 1 : 0) : "memory");
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar_a) : "memory");
            uint32_t done;
            do {
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                             : "=r"(done) : "r"(bar_a) : "memory");
            } while (!done);
            cycles[blockIdx.x] = clock64() - t0;
        }
        __syncwarp();
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tb) : "memory");
}

static cudaError_t rate_of_mma(int sms, long long *d_cycles, long long *h_cycles, double *out)
{
    for (int rep = 0; rep < 2; rep++) gcm_rate_mma_kernel<<<sms, 128, 4096 + 64>>>(d_cycles);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(h_cycles, d_cycles, sizeof(long long) * sms, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return e;
    double sum = 0;
    for (int i = 0; i < sms; i++) sum += (double)h_cycles[i];
    *out = 64.0 * RATE_MMAS / (sum / sms);
    return cudaSuccess;
}

template <int OP>
static cudaError_t rate_of(int sms, uint32_t *sink, long long *d_cycles, long long *h_cycles, double *out)
{
    for (int rep = 0; rep < 2; rep++) gcm_rate_kernel<OP><<<sms, RATE_THREADS>>>(sink, d_cycles, 12345u);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(h_cycles, d_cycles, sizeof(long long) * sms, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return e;
    double sum = 0;
    for (int i = 0; i < sms; i++) sum += (double)h_cycles[i];
    *out = (double)RATE_ITERS * RATE_CHAINS * RATE_THREADS / (sum / sms);
    return cudaSuccess;
}

extern "C" int gcm_measure_pipe_rates(double *rates, int n)
{
    if (!rates || n < GCM_RATE_COUNT) return GCM_ERR_ARG;
    int dev = 0;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    const int sms = prop.multiProcessorCount;
    uint32_t *sink = nullptr;
    long long *d_cycles = nullptr;
    long long *h_cycles = new long long[sms];
    do {
        if ((e = cudaMalloc((void **)&sink, sizeof(uint32_t) * sms * RATE_THREADS)) != cudaSuccess) break;
        if ((e = cudaMalloc((void **)&d_cycles, sizeof(long long) * sms)) != cudaSuccess) break;
        if ((e = rate_of<GCM_RATE_LDS32>(sms, sink, d_cycles, h_cycles, rates + GCM_RATE_LDS32)) != cudaSuccess) break;
        if ((e = rate_of<GCM_RATE_LDS128>(sms, sink, d_cycles, h_cycles, rates + GCM_RATE_LDS128)) != cudaSuccess) break;
        if ((e = rate_of<GCM_RATE_LOP3>(sms, sink, d_cycles, h_cycles, rates + GCM_RATE_LOP3)) != cudaSuccess) break;
        if ((e = rate_of<GCM_RATE_PRMT>(sms, sink, d_cycles, h_cycles, rates + GCM_RATE_PRMT)) != cudaSuccess) break;
        if ((e = rate_of<GCM_RATE_IMAD>(sms, sink, d_cycles, h_cycles, rates + GCM_RATE_IMAD)) != cudaSuccess) break;
        if ((e = rate_of<GCM_RATE_IMAD_WIDE>(sms, sink, d_cycles, h_cycles, rates + GCM_RATE_IMAD_WIDE)) != cudaSuccess) break;
        if ((e = rate_of<GCM_RATE_LOP3_IMAD>(sms, sink, d_cycles, h_cycles, rates + GCM_RATE_LOP3_IMAD)) != cudaSuccess) break;
        if ((e = rate_of_mma(sms, d_cycles, h_cycles, rates + GCM_RATE_MMA_MXF4)) != cudaSuccess) break;
    } while (0);
    if (sink) cudaFree(sink);
    if (d_cycles) cudaFree(d_cycles);
    delete[] h_cycles;
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    return GCM_OK;
}
