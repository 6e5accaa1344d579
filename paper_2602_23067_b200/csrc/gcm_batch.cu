// gcm_batch.cu -- batched many-message entry points (include/gcm.h; SURVEY.md 3.5, 8(a) with the
// per-message rows a1-a3 done 10,000 times for config C4).
//
// Small messages (< BATCH_LARGE_BYTES): ONE persistent kernel, one WARP per message.  A warp takes
// the next message from a ticket counter and runs the whole path on it with no CTA-wide step:
//   a1  key expansion from the lane-replicated round tables (all lanes redundantly: same cost as one)
//   a2  H = E_K(0), the ladder H^(2^k), k = 0..5, by squaring ("table of powers of
//       the hash key H^(2^0), H^(2^1), ..."), and a 4-bit Shoup table of K = H^32 in the warp's own
//       8 KB of shared memory (512 entries: cheap enough to build per message, unlike the 8-bit one)
//   a3  E_K(J0) next to H (lane 0 encrypts 0^128, lane 1 encrypts J0)
//   a4-a7, a10  the row loop shared with the fused kernel (gcm_device.cuh: gcm_rows): cached counter rounds,
//       T-table rounds, XOR, Y <- Y.K xor X with the ciphertext still in registers, the length block as the
//       last virtual block
//   a8  the paper's binary tree (Fig. 3b) across the 32 lanes: at level k the left
//       partial is multiplied by H^(2^k) and XORed into the right one; one more product by H
//   a11  tag, constant-time compare, zero-fill of the output on mismatch.
// Host-descriptor calls (gcm_encrypt_batch / gcm_decrypt_verify_batch): keys never touch global memory except inside
// the descriptor staging, which is wiped after the call.  Device-descriptor calls (gcm_*_batch_device): the caller's
// own gcm_dmsg array is the descriptor array, a kernel orders the tickets, results go into the descriptors.
//
// Large messages (>= BATCH_LARGE_BYTES: FITS-sized HDUs, config C3) are grouped by key and go through
// gcm_multi_kernel (gcm_multi.cu), ONE launch per key with a per-key context that is cached across calls; tags and
// verdicts of both paths come back in one copy.
#include <cuda_runtime.h>
#include <string.h>
#include <stddef.h>
#include <algorithm>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/gcm.h"
#include "gcm_common.cuh"
#include "gcm_device.cuh"
#include "gcm_setup.cuh"
#include "gcm_multi.cuh"
#include "gcm_fused.cuh"
#include "gcm_api_internal.h"

#define BATCH_WARPS        12
#define BATCH_THREADS      (32 * BATCH_WARPS)
#define BATCH_TAB_OFF      AES_TAB_BYTES                 /* per-warp 4-bit tables: 8 KB each */
#define BATCH_TAB_BYTES    8192
#define BATCH_HP_OFF       (BATCH_TAB_OFF + BATCH_WARPS * BATCH_TAB_BYTES)   /* per warp: H^(2^k), k = 0..4 */
#define BATCH_HP_BYTES     128
#define BATCH_SMEM_BYTES   (BATCH_HP_OFF + BATCH_WARPS * BATCH_HP_BYTES)
#define BATCH_LARGE_BYTES  (256ull << 10)                /* at and above: fused kernel per message */

struct BatchDesc {            // one per message, device; == gcm_dmsg of include/gcm.h (the device-descriptor calls hand it over as is)
    uint32_t key[8];
    uint32_t tag[4];          // decrypt: expected tag; device-descriptor encrypt: the tag goes here
    int32_t  status;          // device-descriptor calls: the verdict goes here
    uint32_t key_bits;        // device-descriptor calls: 128 / 256 (the host path sorts by key size itself)
    uint32_t iv[3];
    uint32_t reserved;
    const uint8_t *aad;
    const uint8_t *in;
    uint8_t *out;
    uint64_t aad_len;
    uint64_t len;
};
static_assert(sizeof(BatchDesc) == 112 && sizeof(gcm_dmsg) == 112, "BatchDesc / gcm_dmsg layout");
static_assert(offsetof(BatchDesc, tag) == offsetof(gcm_dmsg, tag) && offsetof(BatchDesc, status) == offsetof(gcm_dmsg, status) &&
              offsetof(BatchDesc, key_bits) == offsetof(gcm_dmsg, key_bits) && offsetof(BatchDesc, iv) == offsetof(gcm_dmsg, iv) &&
              offsetof(BatchDesc, aad) == offsetof(gcm_dmsg, d_aad) && offsetof(BatchDesc, out) == offsetof(gcm_dmsg, d_out) &&
              offsetof(BatchDesc, len) == offsetof(gcm_dmsg, len), "BatchDesc / gcm_dmsg layout");
struct BatchOut {             // where a message's result goes: tag, then verdict
    uint32_t tag[4];
    int status;
};
struct BatchResult {          // one per message, device (host-descriptor path): a BatchOut padded to 32 bytes
    uint32_t tag[4];
    int status;
    int pad[3];
};
static_assert(offsetof(BatchDesc, status) == offsetof(BatchDesc, tag) + 16, "a BatchOut sits inside a BatchDesc");
static_assert(sizeof(BatchResult) == sizeof(MultiResult), "BatchResult / MultiResult layout");

// ---- device ---------------------------------------------------------------------------------------

// y . K through the warp's 4-bit table.  Entry (P, v), P = nibble position 0..31 (nibble P holds the
// coefficients of x^(4P) .. x^(4P+3), highest bit first), is stored at v*512 + (P>>3)*128 + (P&7)*16.
// In step r lane q looks at nibble 8*(r>>3) + ((q + r) & 7): the eight lanes of an LDS.128 phase hit
// eight different 16-byte columns whatever the nibble values are (conflict-free, constant-time).
// rot[k], col[k] (k = r & 7): rotation that brings that nibble to bits 9..12, and the column offset.
__device__ __forceinline__ uint4 ghash_mul4(const uint8_t *tab, const uint32_t (&rot)[8], const uint32_t (&col)[8], uint4 y)
{
    const uint32_t w[4] = {y.x, y.y, y.z, y.w};
    uint4 acc = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int r = 0; r < 32; r++) {
        const uint32_t x = w[r >> 3];
        const uint32_t off = (__funnelshift_r(x, x, rot[r & 7]) & 0x1E00u) | col[r & 7];
        acc = xor4(acc, lds128(tab, off + 128 * (r >> 3)));
    }
    return acc;
}

struct MulK4 {                 // the warp's own 4-bit Shoup table of K (row loop multiplier)
    const uint8_t *tab;
    uint32_t rot[8], col[8];
    __device__ __forceinline__ MulK4(const uint8_t *tab_, uint32_t lane) : tab(tab_)
    {
#pragma unroll
        for (int k = 0; k < 8; k++) {
            const uint32_t n = (lane + k) & 7;
            const uint32_t sh = 8 * (n >> 1) + ((n & 1) ? 0 : 4);    // bit position of the nibble in its word
            rot[k] = (sh - 9) & 31;
            col[k] = n * 16;
        }
    }
    __device__ __forceinline__ uint4 operator()(uint4 y) const { return ghash_mul4(tab, rot, col, y); }
};

__device__ __forceinline__ uint4 shfl4(uint4 v, uint32_t src)
{
    return make_uint4(__shfl_sync(0xFFFFFFFFu, v.x, src), __shfl_sync(0xFFFFFFFFu, v.y, src),
                      __shfl_sync(0xFFFFFFFFu, v.z, src), __shfl_sync(0xFFFFFFFFu, v.w, src));
}

template <int NR, int MODE>
__device__ __forceinline__ void batch_message(const BatchDesc &d, BatchOut *res, const uint8_t *sm,
                                              uint8_t *tab, uint4 *hp, uint32_t lane)
{
    const uint32_t lane4 = lane * 4;
    // a1: key expansion (registers; the same work in every lane)
    uint32_t rk[4 * (NR + 1)];
    aes_key_expand<NR>(sm, lane4, d.key, rk);
    // a2 + a3: lane 0 encrypts 0^128, lane 1 encrypts J0 = IV || 0^31 || 1
    uint4 blk = make_uint4(0, 0, 0, 0);
    if (lane == 1) blk = make_uint4(d.iv[0], d.iv[1], d.iv[2], 0x01000000u);
    blk = aes_encrypt_block<NR>(rk, sm, lane4, blk);
    const uint4 h = shfl4(blk, 0), ekj0 = shfl4(blk, 1);
    // ladder H^(2^k): k = 0..4 kept for the tree, k = 5 is the stride power K
    gf128 hk = gf_from_mem(h);
#pragma unroll 1
    for (int k = 0; k < 5; k++) {
        if (lane == 0) hp[k] = gf_to_mem(hk);
        hk = gf_sqr(hk);
    }
    // 4-bit table of K: lane P owns nibble position P
    {
        gf128 e = gf_zero();
        e.w[lane >> 3] = 1u << (31 - 4 * (lane & 7));            // x^(4P)
        gf128 v0 = gf_mul(e, hk), v1 = gf_mulx(v0), v2 = gf_mulx(v1), v3 = gf_mulx(v2);
        uint4 *row = reinterpret_cast<uint4 *>(tab + (lane >> 3) * 128 + (lane & 7) * 16);
#pragma unroll
        for (int v = 0; v < 16; v++) {
            gf128 a = gf_zero();
            if (v & 8) a = gf_xor(a, v0);
            if (v & 4) a = gf_xor(a, v1);
            if (v & 2) a = gf_xor(a, v2);
            if (v & 1) a = gf_xor(a, v3);
            row[v * 32] = gf_to_mem(a);                          // v * 512 bytes
        }
    }
    __syncwarp();

    // the virtual block sequence [pad | AAD | payload | length block] of the fused kernel, all rows in this warp
    RegMsgView m;
    row_msg_fill(m.r, d.in, d.out, d.aad, d.len, d.aad_len, 0u, 1u, d.len, d.aad_len, false);
    const uint64_t E = m.r.vblocks;
    const uint32_t S = m.r.rows;
    const MulK4 mul(tab, lane);
    const CtrConst cc = ctr_const(rk, d.iv[0], d.iv[1], d.iv[2], sm, lane4);
    const uint4 Y = gcm_rows<NR, MODE>(m, rk, sm, lane, cc, 0u, S, mul);        // a4-a7 (a10: the length block is a row block)

    // a8: the tree over the lanes, in the order of their last blocks (rotate by the ragged remainder):
    // index i = (lane - rem) & 31 holds the partial whose last block is 31 - i blocks before the end.
    const uint32_t rem = (uint32_t)(E - 32ull * (S ? S - 1 : 0)) & 31;      // E mod 32 (0: full last row)
    const uint32_t i = (lane - rem) & 31;
    uint4 Z = Y;
#pragma unroll 1
    for (int k = 0; k < 5; k++) {
        const uint32_t src = ((i - (1u << k)) + rem) & 31;       // lane holding index i - 2^k
        const uint4 left = shfl4(Z, src);
        const uint4 prod = gf_mul_mem(left, hp[k]);
        if ((i & ((2u << k) - 1)) == (2u << k) - 1) Z = xor4(Z, prod);
    }
    // index 31 (lane (31 + rem) & 31) now holds sum X_v . H^(E - 1 - v) with the length block as the last X_v:
    // one more H gives GHASH_H(A, C)
    const uint4 Sg = gf_mul_mem(Z, h);
    const uint4 tag = shfl4(xor4(Sg, ekj0), (31 + rem) & 31);    // a11
    if (MODE == MODE_ENCRYPT) {
        if (lane == 0) {
            res->tag[0] = tag.x; res->tag[1] = tag.y; res->tag[2] = tag.z; res->tag[3] = tag.w;
            res->status = 0;
        }
    } else {
        const uint32_t diff = (tag.x ^ d.tag[0]) | (tag.y ^ d.tag[1]) | (tag.z ^ d.tag[2]) | (tag.w ^ d.tag[3]);
        if (lane == 0) res->status = diff != 0 ? 1 : 0;
        if (diff != 0) {                                        // payload suppression
            __syncwarp();
            const uint64_t len = d.len;
            uint64_t head = (16 - ((uintptr_t)d.out & 15)) & 15;
            if (head > len) head = len;
            const uint64_t mid = (len - head) / 16;
            for (uint64_t k = lane; k < head; k += 32) d.out[k] = 0;
            uint4 *o4 = reinterpret_cast<uint4 *>(d.out + head);
            for (uint64_t k = lane; k < mid; k += 32) o4[k] = make_uint4(0, 0, 0, 0);
            for (uint64_t k = head + mid * 16 + lane; k < len; k += 32) d.out[k] = 0;
        }
    }
}

// order[j]: message index of the j-th ticket (longest first); next: ticket counter.
struct Te0Param { uint32_t w[256]; };      // the round table T0 by value: constant bank, no global load at kernel start

// results: message m's BatchOut is at res_base + m * res_stride (the separate result array of the host-descriptor
// path, or the tag / status fields of the descriptor itself).  n_dev (may be NULL): the ticket count lives on the
// device (written by gcm_batch_order_kernel).
template <int NR, int MODE>
__global__ void __launch_bounds__(BATCH_THREADS, 1)
gcm_batch_kernel(const BatchDesc *descs, uint8_t *res_base, uint32_t res_stride, const uint32_t *order, uint32_t n,
                 const unsigned *n_dev, unsigned *next, const __grid_constant__ Te0Param te0)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t warp = __shfl_sync(0xFFFFFFFFu, threadIdx.x >> 5, 0);
    if (n_dev != nullptr) n = *n_dev;
    if (n == 0) return;
    fill_aes_tables<BATCH_THREADS>(sm, te0.w, threadIdx.x);
    __syncthreads();
    uint8_t *tab = sm + BATCH_TAB_OFF + warp * BATCH_TAB_BYTES;
    uint4 *hp = reinterpret_cast<uint4 *>(sm + BATCH_HP_OFF + warp * BATCH_HP_BYTES);
    for (;;) {
        unsigned j = 0;
        if (lane == 0) j = atomicAdd(next, 1u);
        j = __shfl_sync(0xFFFFFFFFu, j, 0);
        if (j >= n) break;
        const uint32_t m = __ldg(order + j);
        BatchDesc d = descs[m];
        batch_message<NR, MODE>(d, reinterpret_cast<BatchOut *>(res_base + (size_t)m * res_stride), sm, tab, hp, lane);
        __syncwarp();
    }
}

template <int NR, int MODE>
static cudaError_t launch_batch(int blocks, const BatchDesc *descs, uint8_t *res_base, uint32_t res_stride, const uint32_t *order,
                                uint32_t n, const unsigned *n_dev, unsigned *next, const Te0Param &te0, cudaStream_t s)
{
    static std::atomic<bool> configured[GCM_MAX_DEVICES];
    auto kern = gcm_batch_kernel<NR, MODE>;
    cudaError_t e = ensure_smem_attr((const void *)kern, configured, BATCH_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    kern<<<blocks, BATCH_THREADS, BATCH_SMEM_BYTES, s>>>(descs, res_base, res_stride, order, n, n_dev, next, te0);
    return cudaGetLastError();
}

// Device-descriptor calls: ticket order (longest first, by 512-byte rows) for the two key sizes, made on the device.
// One CTA: histogram over (key size, row count), exclusive scan, scatter.  order[0 .. n) holds the AES-128 messages,
// order[n .. 2n) the AES-256 ones; counts[0 / 1] how many of each; descriptors with any other key_bits, a length
// beyond the limits or a NULL buffer get status GCM_ERR_ARG / GCM_ERR_LEN and are left out.  ctr[0..3] = ticket counters and counts, zeroed / written here.
#define ORDER_BUCKETS 514
// What a device-resident descriptor can be refused for before any warp touches it: 0 = take it.  A message longer than
// 2^36 - 32 bytes would wrap the 32-bit counter and reuse keystream (SP 800-38D limit, include/gcm.h); an AAD of 2^36
// bytes or more overflows the 32-bit AAD block count of the row layout; a NULL buffer with a non-zero length would
// fault the launch for every message of the batch.
__device__ __forceinline__ int batch_desc_refusal(const BatchDesc &d)
{
    if (d.key_bits != 128 && d.key_bits != 256) return GCM_ERR_ARG;
    if (d.len > ((1ull << 36) - 32) || d.aad_len >= (1ull << 36)) return GCM_ERR_LEN;
    if ((d.len && (!d.in || !d.out)) || (d.aad_len && !d.aad)) return GCM_ERR_ARG;
    return 0;
}

__global__ void __launch_bounds__(1024, 1)
gcm_batch_order_kernel(BatchDesc *descs, uint32_t n, uint32_t *order, unsigned *ctr)
{
    __shared__ unsigned hist[2][ORDER_BUCKETS];
    __shared__ unsigned total[2];
    const uint32_t t = threadIdx.x;
    for (uint32_t i = t; i < 2 * ORDER_BUCKETS; i += blockDim.x) (&hist[0][0])[i] = 0;
    __syncthreads();
    auto bucket = [](uint64_t len) {          // descending: the longest messages get the lowest bucket
        const uint64_t rows = (len + 511) / 512;
        return (uint32_t)(ORDER_BUCKETS - 1 - (rows < ORDER_BUCKETS - 1 ? rows : ORDER_BUCKETS - 1));
    };
    for (uint32_t i = t; i < n; i += blockDim.x) {
        const int refusal = batch_desc_refusal(descs[i]);
        if (refusal == 0) {
            atomicAdd(&hist[descs[i].key_bits == 256][bucket(descs[i].len)], 1u);
            descs[i].status = GCM_STATUS_PENDING;          // reads "refused" until the message's warp has written it
        } else {
            descs[i].status = refusal;
        }
    }
    __syncthreads();
    if (t < 2) {                               // exclusive scan per key size (514 entries: not worth a parallel scan)
        unsigned run = 0;
        for (int b = 0; b < ORDER_BUCKETS; b++) { const unsigned c = hist[t][b]; hist[t][b] = run; run += c; }
        total[t] = run;
    }
    __syncthreads();
    for (uint32_t i = t; i < n; i += blockDim.x) {
        if (descs[i].status != GCM_STATUS_PENDING) continue;    // refused in the first pass (this thread wrote it)
        const unsigned cls = descs[i].key_bits == 256;
        const unsigned pos = atomicAdd(&hist[cls][bucket(descs[i].len)], 1u);
        order[(size_t)cls * n + pos] = i;
    }
    if (t == 0) { ctr[0] = 0; ctr[1] = 0; ctr[2] = total[0]; ctr[3] = total[1]; }
}

// ---- host -----------------------------------------------------------------------------------------
namespace {

struct BatchState {
    std::mutex mu;
    // fused-path contexts, by key bytes + device
    std::map<std::string, gcm_ctx *> by_key;
    static constexpr size_t kMaxKeys = 64;
    // staging of the small-message path (one device at a time; re-made when the device changes)
    int device = -1;
    int sm_count = 0;
    uint32_t cap = 0;
    BatchDesc *h_desc = nullptr, *d_desc = nullptr;
    BatchResult *h_res = nullptr, *d_res = nullptr;
    uint32_t *h_order = nullptr, *d_order = nullptr;
    unsigned *d_next = nullptr;      // [4]: two ticket counters; the device-descriptor calls add the two ticket counts
    cudaEvent_t dev_done = nullptr;  // last device-descriptor call: its kernels still read the order lists and counters
    bool dev_pending = false;
    uint32_t *d_te0 = nullptr;
    Te0Param h_te0;                  // host copy of the round table (made on the device by gcm_te0_kernel)
    // staging of the large-message path (gcm_multi.cu): descriptors, chunks, per-warp chunk ranges,
    // accumulators + tickets; one pinned block and one device block, grown on demand
    uint8_t *h_multi = nullptr, *d_multi = nullptr;
    size_t multi_cap = 0;
};
BatchState g;

void free_staging_locked()
{
    if (g.device < 0) return;
    DeviceGuard guard(g.device);
    if (g.d_desc) { launch_wipe((uint8_t *)g.d_desc, (uint64_t)g.cap * sizeof(BatchDesc), nullptr, 0); cudaDeviceSynchronize(); cudaFree(g.d_desc); }
    if (g.h_desc) { secure_zero(g.h_desc, (size_t)g.cap * sizeof(BatchDesc)); cudaFreeHost(g.h_desc); }
    if (g.d_res) cudaFree(g.d_res);
    if (g.h_res) cudaFreeHost(g.h_res);
    if (g.d_order) cudaFree(g.d_order);
    if (g.h_order) cudaFreeHost(g.h_order);
    if (g.d_next) cudaFree(g.d_next);
    if (g.dev_done) { cudaEventSynchronize(g.dev_done); cudaEventDestroy(g.dev_done); g.dev_done = nullptr; g.dev_pending = false; }
    if (g.d_te0) cudaFree(g.d_te0);
    if (g.d_multi) cudaFree(g.d_multi);
    if (g.h_multi) cudaFreeHost(g.h_multi);
    g.d_multi = g.h_multi = nullptr; g.multi_cap = 0;
    g.d_desc = g.h_desc = nullptr; g.d_res = g.h_res = nullptr; g.d_order = g.h_order = nullptr;
    g.d_next = nullptr; g.d_te0 = nullptr; g.cap = 0; g.device = -1;
    cudaGetLastError();
}

void evict_keys_locked()
{
    for (auto &kv : g.by_key) gcm_destroy(kv.second);
    // std::string keeps the key bytes: overwrite before the nodes are freed
    for (auto &kv : g.by_key) secure_zero(const_cast<char *>(kv.first.data()), kv.first.size());
    g.by_key.clear();
}

int ensure_staging_locked(uint32_t n)
{
    // one notion of "the device" for the whole library: gcm_set_device's choice, else the caller's current device
    int dev = 0;
    int rc0 = gcm_default_device(&dev);
    if (rc0 != GCM_OK) return rc0;
    cudaError_t e = cudaSuccess;
    if (g.device != dev || g.cap < n) {
        free_staging_locked();
        cudaDeviceProp prop;
        if ((e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) return gcm_cuda_fail(e);
        if ((size_t)prop.sharedMemPerBlockOptin < (size_t)BATCH_SMEM_BYTES) return GCM_ERR_CUDA;
        g.device = dev;
        g.sm_count = prop.multiProcessorCount;
        uint32_t cap = 1024;
        while (cap < n) cap *= 2;
        do {
            if ((e = cudaHostAlloc((void **)&g.h_desc, (size_t)cap * sizeof(BatchDesc), cudaHostAllocDefault)) != cudaSuccess) break;
            if ((e = cudaMalloc((void **)&g.d_desc, (size_t)cap * sizeof(BatchDesc))) != cudaSuccess) break;
            if ((e = cudaHostAlloc((void **)&g.h_res, (size_t)cap * sizeof(BatchResult), cudaHostAllocDefault)) != cudaSuccess) break;
            if ((e = cudaMalloc((void **)&g.d_res, (size_t)cap * sizeof(BatchResult))) != cudaSuccess) break;
            if ((e = cudaHostAlloc((void **)&g.h_order, (size_t)cap * sizeof(uint32_t), cudaHostAllocDefault)) != cudaSuccess) break;
            if ((e = cudaMalloc((void **)&g.d_order, 2 * (size_t)cap * sizeof(uint32_t))) != cudaSuccess) break;   // x 2: the device-descriptor calls keep one list per key size
            if ((e = cudaMalloc((void **)&g.d_next, 4 * sizeof(unsigned))) != cudaSuccess) break;
            if (!g.dev_done && (e = cudaEventCreateWithFlags(&g.dev_done, cudaEventDisableTiming)) != cudaSuccess) break;
            if ((e = cudaMalloc((void **)&g.d_te0, 256 * sizeof(uint32_t))) != cudaSuccess) break;
            launch_te0(g.d_te0, 0);
            if ((e = cudaGetLastError()) != cudaSuccess) break;
            if ((e = cudaMemcpy(g.h_te0.w, g.d_te0, sizeof(g.h_te0.w), cudaMemcpyDeviceToHost)) != cudaSuccess) break;
        } while (0);
        if (e != cudaSuccess) {
            int rc = gcm_cuda_fail(e);
            g.cap = cap;
            free_staging_locked();
            return rc;
        }
        g.cap = cap;
    }
    return GCM_OK;
}

int ctx_for_key_locked(const uint8_t *key, int key_bits, gcm_ctx **out)
{
    std::string id((const char *)key, key_bits / 8);
    id.push_back((char)g.device);
    auto it = g.by_key.find(id);
    if (it != g.by_key.end()) { *out = it->second; secure_zero(&id[0], id.size()); return GCM_OK; }
    gcm_ctx *c = nullptr;
    int rc = gcm_init_on_device(&c, key, key_bits, g.device);
    if (rc == GCM_OK) { g.by_key[id] = c; *out = c; }
    secure_zero(&id[0], id.size());
    return rc;
}

int check_msg(const gcm_msg &m)
{
    if (!m.key || (m.key_bits != 128 && m.key_bits != 256)) return GCM_ERR_ARG;
    if (m.len > ((1ull << 36) - 32) || m.aad_len >= (1ull << 61)) return GCM_ERR_LEN;
    if ((m.aad_len && !m.d_aad) || (m.len && (!m.d_in || !m.d_out))) return GCM_ERR_ARG;
    const uintptr_t a = (uintptr_t)m.d_in, b = (uintptr_t)m.d_out;
    if (m.len && a != b && a < b + m.len && b < a + m.len) return GCM_ERR_ARG;
    return GCM_OK;
}

#define CUB(call)                                                                                  \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) return gcm_cuda_fail(e__);                                         \
    } while (0)

// Large messages (>= BATCH_LARGE_BYTES): grouped by key, ONE launch of gcm_multi_kernel per key (per-key
// context cached across calls).  The rows of all messages of a group are dealt to the warps of the grid in
// contiguous chunks of at most Q = ceil(total rows / warps) rows per warp.
int run_large_locked(gcm_msg *msgs, const std::vector<uint32_t> &large, bool decrypt, cudaStream_t s, int *first_err)
{
    if (large.empty()) return GCM_OK;
    struct Group { gcm_ctx *ctx; std::vector<uint32_t> idx; };
    std::vector<Group> groups;
    std::map<gcm_ctx *, size_t> where;
    for (uint32_t i : large) {
        gcm_ctx *c = nullptr;
        int rc = ctx_for_key_locked(msgs[i].key, msgs[i].key_bits, &c);
        if (rc == GCM_OK && (msgs[i].aad_len + 15) / 16 > 0xFFFFFFFFull) rc = GCM_ERR_LEN;
        if (rc != GCM_OK) { msgs[i].status = rc; if (*first_err == GCM_OK) *first_err = rc; continue; }
        auto it = where.find(c);
        if (it == where.end()) { it = where.emplace(c, groups.size()).first; groups.push_back(Group{c, {}}); }
        groups[it->second].idx.push_back(i);
    }
    if (groups.empty()) return GCM_OK;

    const uint32_t W = (uint32_t)g.sm_count * (MULTI_THREADS / 32);
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    struct Layout { size_t msgs, chunks, wfirst, acc, counter; };
    std::vector<Layout> lay(groups.size());
    size_t total = 0;
    for (size_t k = 0; k < groups.size(); k++) {
        const size_t nk = groups[k].idx.size();
        lay[k].msgs = total;    total += up(nk * sizeof(MultiMsg));
        lay[k].chunks = total;  total += up((nk + W) * sizeof(MultiChunk));
        lay[k].wfirst = total;  total += up((W + 1) * sizeof(uint32_t));
        lay[k].acc = total;     total += up(nk * 16);
        lay[k].counter = total; total += 256;
    }
    if (total > g.multi_cap) {
        cudaStreamSynchronize(s);
        if (g.d_multi) cudaFree(g.d_multi);
        if (g.h_multi) cudaFreeHost(g.h_multi);
        g.d_multi = g.h_multi = nullptr; g.multi_cap = 0;
        size_t cap = 1 << 20;
        while (cap < total) cap *= 2;
        cudaError_t e = cudaHostAlloc((void **)&g.h_multi, cap, cudaHostAllocDefault);
        if (e == cudaSuccess) e = cudaMalloc((void **)&g.d_multi, cap);
        if (e != cudaSuccess) return gcm_cuda_fail(e);
        g.multi_cap = cap;
    }
    memset(g.h_multi, 0, total);

    for (size_t k = 0; k < groups.size(); k++) {
        const std::vector<uint32_t> &idx = groups[k].idx;
        MultiMsg *mm = (MultiMsg *)(g.h_multi + lay[k].msgs);
        MultiChunk *ch = (MultiChunk *)(g.h_multi + lay[k].chunks);
        uint32_t *wf = (uint32_t *)(g.h_multi + lay[k].wfirst);
        uint64_t R = 0;
        for (size_t j = 0; j < idx.size(); j++) {
            const gcm_msg &m = msgs[idx[j]];
            MultiMsg &d = mm[j];
            memcpy(d.iv, m.iv, 12);
            row_msg_fill(d.m, (const uint8_t *)m.d_in, (uint8_t *)m.d_out, (const uint8_t *)m.d_aad, m.len, m.aad_len,
                         0u, 1u, m.len, m.aad_len, false);
            if (decrypt) memcpy(d.tag_expect, m.tag, 16);
            d.result = idx[j];
            R += d.m.rows;
        }
        const uint64_t Q = std::max<uint64_t>(1, (R + W - 1) / W);
        uint32_t w = 0, nch = 0;
        uint64_t budget = Q;
        wf[0] = 0;
        for (size_t j = 0; j < idx.size(); j++) {
            uint32_t r = 0;
            while (r < mm[j].m.rows) {
                const uint32_t take = (uint32_t)std::min<uint64_t>(budget, mm[j].m.rows - r);
                ch[nch].msg = (uint32_t)j; ch[nch].r0 = r; ch[nch].r1 = r + take;
                nch++; r += take; budget -= take;
                if (budget == 0) { wf[++w] = nch; budget = Q; }
            }
        }
        if (wf[w] != nch) wf[++w] = nch;
        const uint32_t n_warps = w;

        MultiParams p;
        memset(&p, 0, sizeof(p));
        gcm_ctx *c = groups[k].ctx;
        memcpy(p.rk, c->h_rk, sizeof(p.rk));
        memcpy(p.te0, c->h_te0, sizeof(p.te0));
        p.tab.te0 = c->d_te0; p.tab.ktab = c->d_ktab; p.tab.hpow = c->d_hpow; p.tab.hx = c->d_hx; p.tab.h = c->d_h;
        p.msgs = (const MultiMsg *)(g.d_multi + lay[k].msgs);
        p.chunks = (const MultiChunk *)(g.d_multi + lay[k].chunks);
        p.warp_first = (const uint32_t *)(g.d_multi + lay[k].wfirst);
        p.n_msgs = (uint32_t)idx.size();
        p.n_warps = n_warps;
        p.acc = (unsigned long long *)(g.d_multi + lay[k].acc);
        p.counter = (unsigned *)(g.d_multi + lay[k].counter);
        p.results = (MultiResult *)g.d_res;
        // one upload per group: descriptors, chunks, chunk ranges and the zeroed accumulators / ticket
        const size_t lo = lay[k].msgs, hi = lay[k].counter + 256;
        CUB(cudaMemcpyAsync(g.d_multi + lo, g.h_multi + lo, hi - lo, cudaMemcpyHostToDevice, s));
        const int blocks = (int)((n_warps + MULTI_THREADS / 32 - 1) / (MULTI_THREADS / 32));
        const MultiMsg *d_msgs = p.msgs;
        cudaError_t e = launch_multi(c->nr, decrypt ? MODE_DECRYPT : MODE_ENCRYPT, blocks, p, s);
        secure_zero(&p, sizeof(p));
        if (e != cudaSuccess) return gcm_cuda_fail(e);
        if (decrypt) {
            launch_multi_wipe(d_msgs, (const MultiResult *)g.d_res, (uint32_t)idx.size(), s);
            CUB(cudaGetLastError());
        }
    }
    return GCM_OK;
}

int run_batch(gcm_msg *msgs, uint32_t n, void *stream, bool decrypt)
{
    if (n && !msgs) return GCM_ERR_ARG;
    if (n == 0) return GCM_OK;
    std::lock_guard<std::mutex> lock(g.mu);
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0;
    int rc = gcm_default_device(&dev);
    if (rc != GCM_OK) return rc;
    DeviceGuard guard(dev);                                 // staging, per-key contexts and kernels all live on `dev`
    CUB(guard.err);
    rc = ensure_staging_locked(n);
    if (rc != GCM_OK) return rc;
    if (g.dev_pending) { CUB(cudaStreamWaitEvent(s, g.dev_done, 0)); g.dev_pending = false; }

    int first_err = GCM_OK;
    std::vector<uint32_t> small[2], large;                  // small[0]: AES-128, small[1]: AES-256
    small[0].reserve(n); small[1].reserve(n);
    for (uint32_t i = 0; i < n; i++) {
        gcm_msg &m = msgs[i];
        m.status = check_msg(m);
        if (m.status != GCM_OK) { if (first_err == GCM_OK) first_err = m.status; continue; }
        BatchDesc &d = g.h_desc[i];
        memset(&d, 0, sizeof(d));
        memcpy(d.key, m.key, m.key_bits / 8);
        memcpy(d.iv, m.iv, 12);
        if (decrypt) memcpy(d.tag, m.tag, 16);
        d.aad = (const uint8_t *)m.d_aad; d.in = (const uint8_t *)m.d_in; d.out = (uint8_t *)m.d_out;
        d.aad_len = m.aad_len; d.len = m.len;
        if (m.len >= BATCH_LARGE_BYTES) large.push_back(i);
        else small[m.key_bits == 256].push_back(i);
    }
    // longest first: the tail of the ticket queue is then made of short messages.  Counting sort on
    // the row count (32 blocks = 512 bytes per row; small messages have at most BATCH_LARGE_BYTES / 512 rows).
    uint32_t pos = 0, start[2], count[2];
    {
        constexpr uint32_t kBuckets = (uint32_t)(BATCH_LARGE_BYTES / 512) + 2;
        std::vector<uint32_t> head(kBuckets + 1);
        for (int k = 0; k < 2; k++) {
            start[k] = pos; count[k] = (uint32_t)small[k].size();
            std::fill(head.begin(), head.end(), 0u);
            auto bucket = [&](uint32_t i) { return kBuckets - 1 - (uint32_t)((msgs[i].len + 511) / 512); };   // descending
            for (uint32_t i : small[k]) head[bucket(i) + 1]++;
            for (uint32_t b = 0; b < kBuckets; b++) head[b + 1] += head[b];
            for (uint32_t i : small[k]) g.h_order[pos + head[bucket(i)]++] = i;
            pos += count[k];
        }
    }
    CUB(cudaMemcpyAsync(g.d_desc, g.h_desc, (size_t)n * sizeof(BatchDesc), cudaMemcpyHostToDevice, s));
    if (pos) CUB(cudaMemcpyAsync(g.d_order, g.h_order, (size_t)pos * sizeof(uint32_t), cudaMemcpyHostToDevice, s));
    CUB(cudaMemsetAsync(g.d_next, 0, 2 * sizeof(unsigned), s));
    // verdicts fail closed: a result slot that no kernel writes reads "refused", never a stale 0 of an earlier call
    if (decrypt) CUB(cudaMemsetAsync(g.d_res, 0xFF, (size_t)n * sizeof(BatchResult), s));
    for (int k = 0; k < 2; k++) {
        if (!count[k]) continue;
        const uint32_t want = (count[k] + BATCH_WARPS - 1) / BATCH_WARPS;
        const int blocks = (int)std::min<uint32_t>(want, (uint32_t)g.sm_count);
        cudaError_t e;
        if (k == 0) e = decrypt ? launch_batch<10, MODE_DECRYPT>(blocks, g.d_desc, (uint8_t *)g.d_res, (uint32_t)sizeof(BatchResult), g.d_order + start[k], count[k], nullptr, g.d_next + k, g.h_te0, s)
                                : launch_batch<10, MODE_ENCRYPT>(blocks, g.d_desc, (uint8_t *)g.d_res, (uint32_t)sizeof(BatchResult), g.d_order + start[k], count[k], nullptr, g.d_next + k, g.h_te0, s);
        else        e = decrypt ? launch_batch<14, MODE_DECRYPT>(blocks, g.d_desc, (uint8_t *)g.d_res, (uint32_t)sizeof(BatchResult), g.d_order + start[k], count[k], nullptr, g.d_next + k, g.h_te0, s)
                                : launch_batch<14, MODE_ENCRYPT>(blocks, g.d_desc, (uint8_t *)g.d_res, (uint32_t)sizeof(BatchResult), g.d_order + start[k], count[k], nullptr, g.d_next + k, g.h_te0, s);
        if (e != cudaSuccess) return gcm_cuda_fail(e);
    }
    rc = run_large_locked(msgs, large, decrypt, s, &first_err);
    if (rc != GCM_OK) return rc;
    CUB(cudaMemcpyAsync(g.h_res, g.d_res, (size_t)n * sizeof(BatchResult), cudaMemcpyDeviceToHost, s));
    // the descriptors hold raw keys: wipe the device copy on the stream, the host copy after the sync
    launch_wipe((uint8_t *)g.d_desc, (uint64_t)n * sizeof(BatchDesc), nullptr, s);
    CUB(cudaGetLastError());
    CUB(cudaStreamSynchronize(s));
    secure_zero(g.h_desc, (size_t)n * sizeof(BatchDesc));
    if (g.by_key.size() > BatchState::kMaxKeys) evict_keys_locked();     // nothing is in flight after the sync
    int failures = 0;
    for (uint32_t i = 0; i < n; i++) {
        gcm_msg &m = msgs[i];
        if (m.status != GCM_OK) continue;
        if (decrypt) {
            m.status = g.h_res[i].status != 0 ? GCM_ERR_AUTH : GCM_OK;
            if (m.status == GCM_ERR_AUTH) failures++;
        } else {
            memcpy(m.tag, g.h_res[i].tag, 16);
        }
    }
    if (first_err != GCM_OK) return first_err;
    return decrypt ? failures : GCM_OK;
}

}  // namespace

// Device-descriptor calls (include/gcm.h: gcm_dmsg): nothing is marshalled on the host.  One small kernel orders the
// tickets, then one persistent warp-per-message kernel per key size; tags and verdicts land in the descriptors.
static int run_batch_device(gcm_dmsg *d_msgs, uint32_t n, void *stream, bool decrypt)
{
    if (n && !d_msgs) return GCM_ERR_ARG;
    if (n == 0) return GCM_OK;
    std::lock_guard<std::mutex> lock(g.mu);
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0;
    int rc = gcm_default_device(&dev);
    if (rc != GCM_OK) return rc;
    DeviceGuard guard(dev);
    CUB(guard.err);
    rc = ensure_staging_locked(n);
    if (rc != GCM_OK) return rc;
    // the previous device-descriptor call may still be reading the order lists and counters
    if (g.dev_pending) CUB(cudaStreamWaitEvent(s, g.dev_done, 0));
    BatchDesc *descs = reinterpret_cast<BatchDesc *>(d_msgs);
    gcm_batch_order_kernel<<<1, 1024, 0, s>>>(descs, n, g.d_order, g.d_next);
    CUB(cudaGetLastError());
    uint8_t *res_base = reinterpret_cast<uint8_t *>(d_msgs) + offsetof(BatchDesc, tag);
    const uint32_t want = (n + BATCH_WARPS - 1) / BATCH_WARPS;
    const int blocks = (int)std::min<uint32_t>(want, (uint32_t)g.sm_count);
    for (int k = 0; k < 2; k++) {
        cudaError_t e;
        const uint32_t *order = g.d_order + (size_t)k * n;
        if (k == 0) e = decrypt ? launch_batch<10, MODE_DECRYPT>(blocks, descs, res_base, (uint32_t)sizeof(BatchDesc), order, n, g.d_next + 2, g.d_next, g.h_te0, s)
                                : launch_batch<10, MODE_ENCRYPT>(blocks, descs, res_base, (uint32_t)sizeof(BatchDesc), order, n, g.d_next + 2, g.d_next, g.h_te0, s);
        else        e = decrypt ? launch_batch<14, MODE_DECRYPT>(blocks, descs, res_base, (uint32_t)sizeof(BatchDesc), order, n, g.d_next + 3, g.d_next + 1, g.h_te0, s)
                                : launch_batch<14, MODE_ENCRYPT>(blocks, descs, res_base, (uint32_t)sizeof(BatchDesc), order, n, g.d_next + 3, g.d_next + 1, g.h_te0, s);
        if (e != cudaSuccess) return gcm_cuda_fail(e);
    }
    CUB(cudaEventRecord(g.dev_done, s));
    g.dev_pending = true;
    return GCM_OK;
}

extern "C" int gcm_encrypt_batch_device(gcm_dmsg *d_msgs, uint32_t n, void *stream) { return run_batch_device(d_msgs, n, stream, false); }
extern "C" int gcm_decrypt_verify_batch_device(gcm_dmsg *d_msgs, uint32_t n, void *stream) { return run_batch_device(d_msgs, n, stream, true); }

extern "C" void gcm_batch_release(void)
{
    std::lock_guard<std::mutex> lock(g.mu);
    evict_keys_locked();
    free_staging_locked();
    gcm_pool_release();
}

extern "C" int gcm_encrypt_batch(gcm_msg *msgs, uint32_t n, void *stream) { return run_batch(msgs, n, stream, false); }
extern "C" int gcm_decrypt_verify_batch(gcm_msg *msgs, uint32_t n, void *stream) { return run_batch(msgs, n, stream, true); }
