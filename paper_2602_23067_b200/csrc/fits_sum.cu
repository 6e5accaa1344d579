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

// ---------------------------------------------------------------------------------------------------
// gfc_datasum_noalloc: the same DATASUM for callers that must not allocate device memory.
//
// gfc_datasum above takes its 8-byte accumulator from cudaMalloc and gives it back with cudaFree on
// every call.  Two kinds of caller cannot live with that:
//   - a process in which another component has already claimed the GPU's memory (a framework's caching
//     allocator sized to the whole HBM, a serving engine that pre-reserved its pools): a raw cudaMalloc
//     there fails with out-of-memory, even for 8 bytes;
//   - a caller in a latency-sensitive loop with other streams in flight (the container's streamH /
//     streamD pair, a collective running beside it): cudaMalloc may, and cudaFree does, wait for the whole
//     device, so an 8-byte allocation stalls work that has nothing to do with the checksum.
// This entry point therefore owns its scratch for the life of the library: a file-scope __device__
// array that the CUDA runtime places in every device's memory when the library's module is loaded
// there and releases at process exit.  Size: GFC_SUM_SCRATCH_WORDS * 8 bytes = 128.25 KiB per GPU.
//
// How the scratch is used.  The data is cut into tiles of GFC_SUM_TILE_BYTES (256 KiB), one CTA each;
// CTA t leaves the sum of its tile in partial[t]; the CTA that draws the last ticket adds the partials
// up, folds the end-around carries and writes the 32-bit DATASUM to the caller's *d_sum.  The array has
// room for GFC_SUM_MAX_TILES (16384) partials, which is where the 4 GiB limit of include/gfc.h comes
// from: a longer buffer is refused with GCM_ERR_LEN before anything is enqueued.
//
//   word 0            ticket counter (must be 0 when a launch starts)
//   words 1 .. 31     unused (keep the partials on their own 256-byte line)
//   words 32 ..       partial[0 .. GFC_SUM_MAX_TILES)
//
// The array is shared by every call on a device and keeps what the last call left in it.  The partials
// need no clearing (each launch overwrites the ones it will read); the ticket counter does, so every
// call enqueues an 8-byte cudaMemsetAsync in front of its kernel (it does not rely on the previous
// launch having finished cleanly).  For the same reason two calls whose kernels can overlap on one GPU
// (different streams without an ordering between them, or two host threads) race on the counter and
// on the partials and give wrong sums: serialise them.
//
// Host code cannot use the name gfc_sum_scratch as a pointer: on the host it is only a handle for the
// symbol (dereferencing or passing it to a kernel reads host memory or faults).  The device address is
// asked for once per device with cudaGetSymbolAddress, while that device is current, and cached.  That
// first call on a device also makes the runtime load the module there, so it should be made once before
// the latency-critical part of the program starts, and before any stream capture is begun.
// ---------------------------------------------------------------------------------------------------
#include <atomic>

#define GFC_SUM_TILE_BYTES    (256u << 10)
#define GFC_SUM_MAX_TILES     16384u
#define GFC_SUM_PARTIALS_AT   32u
#define GFC_SUM_SCRATCH_WORDS (GFC_SUM_PARTIALS_AT + GFC_SUM_MAX_TILES)
#define GFC_SUM_MAX_DEVICES   64       /* devices whose scratch address is cached; beyond: looked up per call */

static_assert((uint64_t)GFC_SUM_TILE_BYTES * GFC_SUM_MAX_TILES == GFC_DATASUM_NOALLOC_MAX_BYTES,
              "include/gfc.h states the limit that the scratch array can serve");

static __device__ __align__(256) unsigned long long gfc_sum_scratch[GFC_SUM_SCRATCH_WORDS];

// CTA-wide sum of s; the result is valid in thread 0.  `red` holds one word per warp.
__device__ __forceinline__ unsigned long long cta_sum(unsigned long long s, unsigned long long *red)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = threadIdx.x < SUM_THREADS / 32 ? red[threadIdx.x] : 0ull;
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    }
    __syncthreads();                       // red may be reused by the caller
    return s;
}

// One CTA per 256 KiB tile; gridDim.x = number of tiles <= GFC_SUM_MAX_TILES.  scratch: the device
// address of gfc_sum_scratch (word 0 zeroed by the memset enqueued in front of this launch).
__global__ void __launch_bounds__(SUM_THREADS)
fits_sum32_tiles_kernel(const uint8_t *__restrict__ p, uint64_t nbytes, unsigned long long *scratch,
                        uint32_t *__restrict__ d_sum)
{
    __shared__ unsigned long long red[SUM_THREADS / 32];
    __shared__ unsigned last;
    constexpr uint32_t TILE16 = GFC_SUM_TILE_BYTES / 16;
    const uint64_t n16 = nbytes / 16;
    const uint4 *v = reinterpret_cast<const uint4 *>(p);
    const uint64_t lo = (uint64_t)blockIdx.x * TILE16;
    const uint64_t hi = lo + TILE16 < n16 ? lo + TILE16 : n16;
    unsigned long long s0 = 0, s1 = 0;
    uint64_t i = lo + threadIdx.x;
    // four loads in flight per thread and iteration
    for (; i + 3 * SUM_THREADS < hi; i += 4 * SUM_THREADS) {
        const uint4 a = __ldcs(v + i), b = __ldcs(v + i + SUM_THREADS);
        const uint4 c = __ldcs(v + i + 2 * SUM_THREADS), d = __ldcs(v + i + 3 * SUM_THREADS);
        s0 += (unsigned long long)be32(a.x) + be32(a.y) + be32(a.z) + be32(a.w);
        s1 += (unsigned long long)be32(b.x) + be32(b.y) + be32(b.z) + be32(b.w);
        s0 += (unsigned long long)be32(c.x) + be32(c.y) + be32(c.z) + be32(c.w);
        s1 += (unsigned long long)be32(d.x) + be32(d.y) + be32(d.z) + be32(d.w);
    }
    for (; i < hi; i += SUM_THREADS) {
        const uint4 a = __ldcs(v + i);
        s0 += (unsigned long long)be32(a.x) + be32(a.y) + be32(a.z) + be32(a.w);
    }
    // ragged tail (< 16 bytes) belongs to the last tile; missing bytes count as zero
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        for (uint64_t b = n16 * 16; b < nbytes; b++)
            s1 += (unsigned long long)p[b] << (8 * (3 - (b & 3)));
    }
    unsigned long long s = cta_sum(fold33(s0) + fold33(s1), red);
    if (threadIdx.x == 0) {
        scratch[GFC_SUM_PARTIALS_AT + blockIdx.x] = fold33(s);
        __threadfence();                                         // the partial is visible before the ticket is
        last = atomicAdd(reinterpret_cast<unsigned *>(scratch), 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    // the CTA with the last ticket: every partial of this launch has been published
    __threadfence();
    s = 0;
    for (uint32_t t = threadIdx.x; t < gridDim.x; t += SUM_THREADS)
        s += __ldcg(scratch + GFC_SUM_PARTIALS_AT + t);          // L2: written by other SMs
    s = cta_sum(s, red);
    if (threadIdx.x == 0) {
        while (s >> 32) s = (s & 0xFFFFFFFFull) + (s >> 32);     // end-around carry
        *d_sum = (uint32_t)s;
        scratch[0] = 0;                                          // leave the counter as it was found
    }
}

// Device address of gfc_sum_scratch on the CURRENT device `dev`, looked up once per device.
static cudaError_t sum_scratch_address(int dev, unsigned long long **out)
{
    static std::atomic<unsigned long long *> cache[GFC_SUM_MAX_DEVICES];
    const bool tracked = dev >= 0 && dev < GFC_SUM_MAX_DEVICES;
    unsigned long long *ptr = tracked ? cache[dev].load(std::memory_order_acquire) : nullptr;
    if (!ptr) {
        // gfc_sum_scratch is passed as the symbol's handle here, never as an address
        const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, gfc_sum_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        if (tracked) cache[dev].store(ptr, std::memory_order_release);   // two threads would store the same value
    }
    *out = ptr;
    return cudaSuccess;
}

extern "C" int gfc_datasum_noalloc(const void *d_data, uint64_t len, uint32_t *d_sum, void *cuda_stream)
{
    if (!d_sum || (len && !d_data) || ((uintptr_t)d_data & 15) || ((uintptr_t)d_sum & 3)) return GCM_ERR_ARG;
    if (len > GFC_DATASUM_NOALLOC_MAX_BYTES) return GCM_ERR_LEN;       // more tiles than the scratch has partials
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (len == 0) {                                                      // the sum of nothing; no scratch involved
        e = cudaMemsetAsync(d_sum, 0, sizeof(uint32_t), s);
        return e == cudaSuccess ? GCM_OK : gcm_cuda_fail(e);
    }
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return gcm_cuda_fail(e);   // the data lives on the current device
    unsigned long long *scratch = nullptr;
    if ((e = sum_scratch_address(dev, &scratch)) != cudaSuccess) return gcm_cuda_fail(e);
    const unsigned tiles = (unsigned)((len + GFC_SUM_TILE_BYTES - 1) / GFC_SUM_TILE_BYTES);
    if ((e = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), s)) != cudaSuccess) return gcm_cuda_fail(e);
    fits_sum32_tiles_kernel<<<tiles, SUM_THREADS, 0, s>>>((const uint8_t *)d_data, len, scratch, d_sum);
    e = cudaGetLastError();
    return e == cudaSuccess ? GCM_OK : gcm_cuda_fail(e);
}
