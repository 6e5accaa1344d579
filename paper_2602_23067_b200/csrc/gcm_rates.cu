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
    } while (0);
    if (sink) cudaFree(sink);
    if (d_cycles) cudaFree(d_cycles);
    delete[] h_cycles;
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    return GCM_OK;
}
