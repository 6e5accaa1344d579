// fits_sum.cu -- DATASUM of a device-resident data unit: the 1's-complement sum of its big-endian
// 32-bit words (FITS checksum convention, cited by the paper at PAPER.md L135: the container "writes
// the FITS-standard CHECKSUM and DATASUM keywords to both HDUs").
//
// HBM-bound: one 16-byte load per thread and iteration (coalesced, streaming), four byte swaps and
// four 64-bit adds; algorithmic traffic 1 byte read per byte.  1's-complement addition is ordinary
// addition with the carries folded back in, and it is associative and commutative, so the words may be
// summed in any order in 64-bit accumulators and folded at the end.  Persistent grid (a multiple of the
// SM count), grid-stride loop, shuffle + shared-memory reduction, one atomicAdd per CTA.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gfc.h"
#include "gcm_api_internal.h"
#include "fits_sum.cuh"

#define SUM_THREADS 512

__device__ __forceinline__ uint32_t be32(uint32_t w) { return __byte_perm(w, 0, 0x0123); }

// fold a 64-bit partial to at most 33 bits (keeps the value modulo 2^32 - 1, which is all that matters)
__device__ __forceinline__ unsigned long long fold33(unsigned long long s)
{
    return (s & 0xFFFFFFFFull) + (s >> 32);
}

__global__ void __launch_bounds__(SUM_THREADS)
fits_sum32_kernel(const uint8_t *__restrict__ p, uint64_t nbytes, unsigned long long *acc)
{
    __shared__ unsigned long long red[SUM_THREADS / 32];
    const uint64_t n16 = nbytes / 16;
    const uint4 *v = reinterpret_cast<const uint4 *>(p);
    unsigned long long s0 = 0, s1 = 0;
    const uint64_t stride = (uint64_t)gridDim.x * SUM_THREADS;
    uint64_t i = (uint64_t)blockIdx.x * SUM_THREADS + threadIdx.x;
    // two loads in flight per thread and iteration
    for (; i + stride < n16; i += 2 * stride) {
        const uint4 a = __ldcs(v + i), b = __ldcs(v + i + stride);
        s0 += (unsigned long long)be32(a.x) + be32(a.y) + be32(a.z) + be32(a.w);
        s1 += (unsigned long long)be32(b.x) + be32(b.y) + be32(b.z) + be32(b.w);
    }
    if (i < n16) {
        const uint4 a = __ldcs(v + i);
        s0 += (unsigned long long)be32(a.x) + be32(a.y) + be32(a.z) + be32(a.w);
    }
    // ragged tail (< 16 bytes): missing bytes count as zero (the data unit is zero-padded to 2880)
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        for (uint64_t b = n16 * 16; b < nbytes; b++)
            s1 += (unsigned long long)p[b] << (8 * (3 - (b & 3)));
    }
    unsigned long long s = fold33(s0) + fold33(s1);
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = threadIdx.x < SUM_THREADS / 32 ? red[threadIdx.x] : 0ull;
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
        if (threadIdx.x == 0) atomicAdd(acc, fold33(s));
    }
}

cudaError_t launch_fits_sum32(const uint8_t *d_data, uint64_t nbytes, unsigned long long *d_acc, int sm_count,
                              cudaStream_t s)
{
    if (nbytes == 0) return cudaSuccess;
    const uint64_t n16 = nbytes / 16;
    uint64_t want = (n16 + 2ull * SUM_THREADS - 1) / (2ull * SUM_THREADS);
    const uint64_t cap = (uint64_t)sm_count * 4;          // 4 resident CTAs of 512 threads per SM
    int grid = (int)(want < 1 ? 1 : (want > cap ? cap : want));
    fits_sum32_kernel<<<grid, SUM_THREADS, 0, s>>>(d_data, nbytes, d_acc);
    return cudaGetLastError();
}

uint32_t fits_sum_fold(unsigned long long s)
{
    while (s >> 32) s = (s & 0xFFFFFFFFull) + (s >> 32);
    return (uint32_t)s;
}

extern "C" int gfc_datasum_async(const void *d_data, uint64_t len, void *d_acc, void *cuda_stream)
{
    if (!d_acc || (len && !d_data) || ((uintptr_t)d_data & 15) || ((uintptr_t)d_acc & 7)) return GCM_ERR_ARG;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);            // the data lives on the caller's current device
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    const int rc = gcm_sm_count(dev, &sms);        // cached per device
    if (rc != GCM_OK) return rc;
    e = launch_fits_sum32((const uint8_t *)d_data, len, (unsigned long long *)d_acc, sms, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? GCM_OK : gcm_cuda_fail(e);
}

extern "C" int gfc_datasum(const void *d_data, uint64_t len, uint32_t *sum, void *cuda_stream)
{
    if (!sum || (len && !d_data) || ((uintptr_t)d_data & 15)) return GCM_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    unsigned long long *d_acc = nullptr, h = 0;
    if ((e = cudaMalloc((void **)&d_acc, 8)) != cudaSuccess) return gcm_cuda_fail(e);
    do {
        if ((e = cudaMemsetAsync(d_acc, 0, 8, s)) != cudaSuccess) break;
        if ((e = launch_fits_sum32((const uint8_t *)d_data, len, d_acc, sms, s)) != cudaSuccess) break;
        if ((e = cudaMemcpyAsync(&h, d_acc, 8, cudaMemcpyDeviceToHost, s)) != cudaSuccess) break;
        e = cudaStreamSynchronize(s);
    } while (0);
    cudaFree(d_acc);
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    *sum = fits_sum_fold(h);
    return GCM_OK;
}
