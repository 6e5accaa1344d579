// gcm_api.cu -- the C ABI of libb200gcm.so (include/gcm.h): argument checks, launch parameters,
// context ownership.  No arithmetic of the method runs on the host: key schedule, H, powers,
// CTR, GHASH, tag and compare are all kernels (gcm_setup.cu, gcm_fused.cu, gcm_batch.cu).
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>
#include <stdlib.h>
#include <stddef.h>
#include <atomic>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/gcm.h"
#include "gcm_common.cuh"
#include "gcm_setup.cuh"
#include "gcm_fused.cuh"
#include "gcm_tc.cuh"
#include "gcm_api_internal.h"

// Device for new contexts: -1 = the calling thread's current CUDA device, else the ordinal given to gcm_set_device.
static std::atomic<int> g_device{-1};
static std::atomic<int> g_last_cuda_error{0};

// Wiped (device slab, pinned block) pairs of destroyed contexts, kept for the next gcm_init on the same
// device: cudaMalloc + cudaHostAlloc cost milliseconds, the setup kernel 56 us (the paper pre-allocates
// once per session for the same reason).  At most kPoolMax pairs are kept.
namespace {
struct PooledSlab { int device; uint8_t *d_slab; size_t bytes; };
constexpr size_t kPoolMax = 4;
std::mutex g_pool_mu;
std::vector<PooledSlab> g_pool;

// 64-byte blocks of mapped pinned memory (tag / verdict of the synchronous calls) come out of one page that
// is allocated once per process: a cudaHostAlloc per context costs about two milliseconds.
uint8_t *g_pin_page = nullptr;
uint64_t g_pin_used = 0;

uint8_t *pin_take()
{
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (!g_pin_page && cudaHostAlloc((void **)&g_pin_page, 64 * 64, cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess) {
        g_pin_page = nullptr;
        cudaGetLastError();
    }
    if (g_pin_page)
        for (int i = 0; i < 64; i++)
            if (!(g_pin_used >> i & 1)) { g_pin_used |= 1ull << i; return g_pin_page + 64 * i; }
    uint8_t *p = nullptr;                                  // page exhausted (more than 64 live contexts)
    if (cudaHostAlloc((void **)&p, 64, cudaHostAllocMapped) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}

void pin_give(uint8_t *p)
{
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (g_pin_page && p >= g_pin_page && p < g_pin_page + 64 * 64) g_pin_used &= ~(1ull << ((p - g_pin_page) / 64));
    else cudaFreeHost(p);
}
}

int gcm_cuda_fail(cudaError_t e)
{
    g_last_cuda_error.store((int)e);
    cudaGetLastError();   // clear the sticky-free error state
    return e == cudaErrorMemoryAllocation ? GCM_ERR_NOMEM : GCM_ERR_CUDA;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) return gcm_cuda_fail(e__);                                         \
    } while (0)

extern "C" const char *gcm_version(void) { return "b200gcm 0.2 sm_100a"; }

extern "C" int gcm_set_device(int ordinal)
{
    int count = 0;
    CU(cudaGetDeviceCount(&count));
    if (ordinal < -1 || ordinal >= count) return GCM_ERR_ARG;
    g_device.store(ordinal);        // the caller's current device is left alone
    return GCM_OK;
}

int gcm_default_device(int *device)
{
    const int d = g_device.load();
    if (d >= 0) { *device = d; return GCM_OK; }
    CU(cudaGetDevice(device));
    return GCM_OK;
}

// SM count per device, queried once (cudaDeviceGetAttribute is cheap, but this sits on the latency path)
int gcm_sm_count(int device, int *sms)
{
    static std::atomic<int> cache[GCM_MAX_DEVICES];
    if (device >= 0 && device < GCM_MAX_DEVICES && cache[device].load(std::memory_order_relaxed) > 0) {
        *sms = cache[device].load(std::memory_order_relaxed);
        return GCM_OK;
    }
    CU(cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, device));
    if (device >= 0 && device < GCM_MAX_DEVICES) cache[device].store(*sms, std::memory_order_relaxed);
    return GCM_OK;
}

extern "C" int gcm_last_cuda_error(void) { return g_last_cuda_error.load(); }
extern "C" const char *gcm_last_cuda_error_string(void)
{
    return cudaGetErrorString((cudaError_t)g_last_cuda_error.load());
}

static SetupParams setup_params(gcm_ctx *c, const uint8_t *key)
{
    SetupParams sp;
    memset(&sp, 0, sizeof(sp));
    if (key) memcpy(sp.key, key, c->key_bits / 8);
    sp.key_bits = c->key_bits;
    sp.te0 = c->d_te0;
    sp.rk = c->d_rk;
    sp.h = c->d_h;
    sp.hpow = c->d_hpow;
    sp.hx = c->d_hx;
    sp.ktab = c->d_ktab;
    return sp;
}

extern "C" int gcm_init(gcm_ctx **out, const uint8_t *key, int key_bits)
{
    if (!out) return GCM_ERR_ARG;
    *out = nullptr;
    if (!key || (key_bits != 128 && key_bits != 256)) return GCM_ERR_ARG;     // before any CUDA call
    int device = 0;
    int rc = gcm_default_device(&device);
    if (rc != GCM_OK) return rc;
    return gcm_init_on_device(out, key, key_bits, device);
}

int gcm_init_on_device(gcm_ctx **out, const uint8_t *key, int key_bits, int device)
{
    if (!out || !key || (key_bits != 128 && key_bits != 256)) return GCM_ERR_ARG;
    *out = nullptr;
    DeviceGuard guard(device);
    CU(guard.err);
    // two attribute queries, not cudaGetDeviceProperties (which takes milliseconds)
    int sm_count = 0, smem_optin = 0;
    CU(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, device));
    CU(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
    if ((size_t)smem_optin < (size_t)FUSED_SMEM_BYTES) return GCM_ERR_CUDA;

    gcm_ctx *c = new (std::nothrow) gcm_ctx();      // value-initialised: every member zero
    if (!c) return GCM_ERR_NOMEM;
    c->device = device;
    c->key_bits = key_bits;
    c->nr = key_bits == 128 ? 10 : 14;
    c->sm_count = sm_count;
    c->grid = c->sm_count;
    c->threads = GCM_MAX_THREADS;
    c->engine = GCM_GHASH_AUTO;

    // one slab for all device-side state
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
    size_t o_te0 = take(256 * 4), o_rk = take(64 * 4), o_h = take(16);
    size_t o_hpow = take((GCM_STRIDE + 1) * 16), o_hx = take(HX_ENTRIES * 16);
    size_t o_ktab = take(KTAB_BYTES), o_part = take(GCM_MAX_GRID * 16);
    size_t o_cnt = take(4), o_tag = take(16), o_status = take(4), o_bmat = take(TC_BMAT_TOTAL);
    size_t o_bmat2 = take(GT_BMAT_TOTAL), o_ktab2 = take(KTAB_BYTES), o_gt = take(128);   // d_gt[0..2]: chain state; bytes 64..95: clock probe of gcm_tc2_kernel
    c->slab_bytes = off;
    cudaError_t e = cudaSuccess;
    {
        std::lock_guard<std::mutex> lock(g_pool_mu);
        for (size_t i = 0; i < g_pool.size(); i++)
            if (g_pool[i].device == device && g_pool[i].bytes == c->slab_bytes) {
                c->d_slab = g_pool[i].d_slab;
                g_pool.erase(g_pool.begin() + i);
                break;
            }
    }
    if (!c->d_slab) e = cudaMalloc((void **)&c->d_slab, c->slab_bytes);
    if (e != cudaSuccess) { delete c; return gcm_cuda_fail(e); }
    c->d_te0 = (uint32_t *)(c->d_slab + o_te0);
    c->d_rk = (uint32_t *)(c->d_slab + o_rk);
    c->d_h = (uint4 *)(c->d_slab + o_h);
    c->d_hpow = (uint4 *)(c->d_slab + o_hpow);
    c->d_hx = (uint4 *)(c->d_slab + o_hx);
    c->d_ktab = (uint4 *)(c->d_slab + o_ktab);
    c->d_partials = (uint4 *)(c->d_slab + o_part);
    c->d_counter = (unsigned *)(c->d_slab + o_cnt);
    c->d_tag = (uint4 *)(c->d_slab + o_tag);
    c->d_status = (int *)(c->d_slab + o_status);
    c->d_bmat = (uint4 *)(c->d_slab + o_bmat);
    c->d_bmat2 = (uint4 *)(c->d_slab + o_bmat2);
    c->d_ktab2 = (uint4 *)(c->d_slab + o_ktab2);
    c->d_gt = (uint4 *)(c->d_slab + o_gt);

    int rc = GCM_OK;
    do {
        if ((c->h_pinned = pin_take()) == nullptr) { e = cudaErrorMemoryAllocation; break; }
        if ((e = cudaMemsetAsync(c->d_slab, 0, c->slab_bytes, 0)) != cudaSuccess) break;
        SetupParams sp = setup_params(c, key);
        launch_setup(sp, 0);
        secure_zero(&sp, sizeof(sp));
        launch_tc_setup(c->d_hx, c->d_bmat, 0);        // a2 for the tensor-core GHASH: bit matrices of K^0 .. K^TC_L
        launch_ghash_tc_setup(c->d_hx, c->d_bmat2, c->d_ktab2, 0);
        if ((e = cudaGetLastError()) != cudaSuccess) break;
        // synchronous copy: the tables are complete before any kernel of this context can be launched (the
        // fused kernel reads them ahead of griddepcontrol.wait and relies on that)
        static_assert(offsetof(gcm_ctx, h_rk) == offsetof(gcm_ctx, h_te0) + 1024, "h_te0 and h_rk are adjacent");
        if ((e = cudaMemcpy(c->h_te0, c->d_te0, sizeof(c->h_te0) + sizeof(c->h_rk), cudaMemcpyDeviceToHost)) != cudaSuccess) break;
    } while (0);
    if (e != cudaSuccess) {
        rc = gcm_cuda_fail(e);
        gcm_destroy(c);
        return rc;
    }
    *out = c;
    return GCM_OK;
}

extern "C" void gcm_destroy(gcm_ctx *c)
{
    if (!c) return;
    DeviceGuard guard(c->device);
    gcm_host_pipe_free(c);
    bool pooled = false;
    if (c->d_slab) {
        launch_wipe(c->d_slab, c->slab_bytes, nullptr, 0);      // key material never outlives the context
        cudaDeviceSynchronize();
    }
    if (c->h_pinned) {
        secure_zero(c->h_pinned, 64);
        pin_give(c->h_pinned);
    }
    if (c->d_slab && cudaGetLastError() == cudaSuccess) {
        std::lock_guard<std::mutex> lock(g_pool_mu);
        if (g_pool.size() < kPoolMax) {
            g_pool.push_back(PooledSlab{c->device, c->d_slab, c->slab_bytes});
            pooled = true;
        }
    }
    if (!pooled && c->d_slab) cudaFree(c->d_slab);
    cudaGetLastError();
    secure_zero(c->h_rk, sizeof(c->h_rk));
    delete c;
}

void gcm_pool_release(void)
{
    std::lock_guard<std::mutex> lock(g_pool_mu);
    for (const PooledSlab &p : g_pool) {           // already wiped when they were pooled
        DeviceGuard guard(p.device);
        cudaFree(p.d_slab);
    }
    g_pool.clear();
    if (g_pin_page && g_pin_used == 0) {
        cudaFreeHost(g_pin_page);
        g_pin_page = nullptr;
    }
    cudaGetLastError();
}

extern "C" int gcm_set_geometry(gcm_ctx *c, int grid, int threads)
{
    if (!c) return GCM_ERR_ARG;
    if (grid == 0) grid = c->sm_count;
    if (threads == 0) threads = GCM_MAX_THREADS;
    if (grid < 1 || grid > GCM_MAX_GRID || (threads != 256 && threads != 384 && threads != 512)) return GCM_ERR_ARG;
    // no table depends on the geometry: the GHASH stride power is H^32 for every launch shape
    c->grid = grid;
    c->threads = threads;
    return GCM_OK;
}

extern "C" int gcm_set_ghash_engine(gcm_ctx *c, int engine)
{
    if (!c || (engine != GCM_GHASH_TABLE && engine != GCM_GHASH_TENSOR && engine != GCM_GHASH_AUTO)) return GCM_ERR_ARG;
    c->engine = engine;
    return GCM_OK;
}

extern "C" int gcm_get_ghash_engine(const gcm_ctx *c, int *engine)
{
    if (!c || !engine) return GCM_ERR_ARG;
    *engine = c->engine;
    return GCM_OK;
}

extern "C" int gcm_get_geometry(const gcm_ctx *c, int *grid, int *threads)
{
    if (!c) return GCM_ERR_ARG;
    if (grid) *grid = c->grid;
    if (threads) *threads = c->threads;
    return GCM_OK;
}

extern "C" int gcm_get_hash_subkey(const gcm_ctx *c, uint8_t h[16])
{
    if (!c || !h) return GCM_ERR_ARG;
    DeviceGuard guard(c->device);
    CU(guard.err);
    CU(cudaMemcpy(h, c->d_h, 16, cudaMemcpyDeviceToHost));
    return GCM_OK;
}

extern "C" int gcm_debug_row_layout(uint64_t len, uint64_t aad_len, uint32_t ctr_base, int last, int aligned, gcm_row_layout *out)
{
    if (!out) return GCM_ERR_ARG;
    if (len > ((1ull << 36) - 32) || aad_len >= (1ull << 61) || (aad_len + 15) / 16 > 0xFFFFFFFFull) return GCM_ERR_LEN;
    RowMsg m;
    memset(&m, 0, sizeof(m));
    // only the alignment of the pointers matters to the layout
    const uint8_t *fake = (const uint8_t *)(uintptr_t)(aligned ? 0x1000 : 0x1001);
    row_msg_fill(m, fake, (uint8_t *)(uintptr_t)fake, fake, len, aad_len, ctr_base, last ? 1u : 0u, len, aad_len, false);
    if (m.vblocks >= GCM_MAX_VBLOCKS) return GCM_ERR_LEN;
    memset(out, 0, sizeof(*out));
    out->vblocks = m.vblocks; out->base = m.base; out->pad = m.pad; out->n_aad_blocks = m.n_aad_blocks;
    out->rows = m.rows; out->fast_lo = m.fast_lo; out->fast_hi = m.fast_hi; out->ctr_delta = m.ctr_delta;
    out->len_block = m.len_block;
    return GCM_OK;
}

extern "C" int gcm_set_phase_stamps(gcm_ctx *c, void *d_stamps)
{
    if (!c) return GCM_ERR_ARG;
    c->d_stamps = (unsigned long long *)d_stamps;
    return GCM_OK;
}

// Argument checks and launch parameters common to encrypt / decrypt / ghash (see gcm_api_internal.h).
int gcm_build_params(gcm_ctx *c, int mode, const uint8_t *iv, const void *d_aad, uint64_t aad_len,
                     const void *d_in, uint64_t len, void *d_out, uint32_t ctr_base, bool last,
                     uint64_t final_len, uint64_t final_aad_len, GcmParams *p, int *blocks)
{
    if (!c) return GCM_ERR_ARG;
    if (mode != MODE_GHASH && !iv) return GCM_ERR_ARG;
    if (len > ((1ull << 36) - 32) || aad_len >= (1ull << 61)) return GCM_ERR_LEN;
    if ((aad_len && !d_aad) || (len && !d_in)) return GCM_ERR_ARG;
    if (mode != MODE_GHASH && len && !d_out) return GCM_ERR_ARG;
    const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
    if (mode != MODE_GHASH && len && a != b && a < b + len && b < a + len) return GCM_ERR_ARG;  // partial overlap
    if ((aad_len + 15) / 16 > 0xFFFFFFFFull) return GCM_ERR_LEN;

    memset(p, 0, sizeof(*p));
    row_msg_fill(p->m, (const uint8_t *)d_in, (uint8_t *)d_out, (const uint8_t *)d_aad, len, aad_len, ctr_base,
                 last ? 1u : 0u, final_len, final_aad_len, mode == MODE_GHASH);
    if (p->m.vblocks >= GCM_MAX_VBLOCKS) return GCM_ERR_LEN;
    memcpy(p->rk, c->h_rk, sizeof(p->rk));
    memcpy(p->te0, c->h_te0, sizeof(p->te0));
    if (iv) memcpy(p->iv, iv, 12);
    // rows are dealt to the warps of the grid in contiguous runs balanced to +-1 row; a short message uses
    // only as many CTAs as it has rows for
    const uint64_t S = p->m.rows;
    const uint64_t wpc = c->engine == GCM_GHASH_TENSOR ? TC_PRODUCER_WARPS : (uint64_t)c->threads / 32;   // warps per CTA that take rows
    uint64_t want = (S + wpc - 1) / wpc;
    if (want < 1) want = 1;
    if (want > (uint64_t)c->grid) want = (uint64_t)c->grid;
    *blocks = (int)want;
    p->warps = (uint32_t)(want * wpc);
    p->tab.te0 = c->d_te0;
    p->tab.ktab = c->d_ktab;
    p->tab.hpow = c->d_hpow;
    p->tab.hx = c->d_hx;
    p->tab.h = c->d_h;
    p->tab.bmat = c->d_bmat;
    p->partials = c->d_partials;
    p->counter = c->d_counter;
    c->ticket_next += (unsigned)want;                            // epoch scheme: see GcmParams::ticket_last
    p->ticket_last = c->ticket_next - 1;
    p->tag_out = c->d_tag;
    p->status = c->d_status;
    p->stamps = c->d_stamps;
    return GCM_OK;
}

// Header-sized messages take the single-CTA latency kernel (gcm_small.cu) under the default geometry; an
// explicit gcm_set_geometry always selects the fused kernel (the geometry tests rely on that).
cudaError_t gcm_launch_fused(gcm_ctx *c, int mode, int blocks, const GcmParams &p, cudaStream_t s)
{
    const cudaError_t e = c->engine == GCM_GHASH_TENSOR ? launch_tc(c->nr, mode, blocks, p, s)
                                                        : launch_fused(c->nr, mode, c->threads, blocks, p, s);
    if (e != cudaSuccess) c->ticket_next -= (unsigned)blocks;    // the launch was not made: its tickets are not drawn
    return e;
}

static cudaError_t launch_auto(gcm_ctx *c, int mode, int blocks, GcmParams &p, cudaStream_t s)
{
    const uint64_t n_ghash = (uint64_t)p.m.n_aad_blocks + (p.m.len + 15) / 16 + 1;
    if (mode != MODE_GHASH && n_ghash <= SMALL_MAX_BLOCKS && c->grid == c->sm_count && c->threads == GCM_MAX_THREADS &&
        !p.chain_in && !p.chain_out) {
        c->ticket_next -= (unsigned)blocks;                      // no tickets are drawn by the latency kernel
        return launch_small(c->nr, mode, p, s);
    }
    return gcm_launch_fused(c, mode, blocks, p, s);
}

#define LOCK_CTX(c)                                                                                \
    if (!(c)) return GCM_ERR_ARG;                                                                  \
    CtxLock lock__(c);                                                                             \
    if (!lock__.ok) return GCM_ERR_BUSY;                                                           \
    DeviceGuard guard__((c)->device);                                                              \
    CU(guard__.err)

// What the launch that FINISHES a message needs besides the common parameters.
struct FinalOpts {
    uint4 *tag_out;             // encrypt: device (or mapped host) tag
    const uint4 *tag_in;        // decrypt: device tag, or NULL -> tag_expect
    const uint8_t *tag_expect;  // decrypt: 16 bytes by value, or NULL
    int *status;                // decrypt: verdict word
    uint32_t status_init;
};

static void apply_final(GcmParams &p, const FinalOpts &f)
{
    if (f.tag_out) p.tag_out = f.tag_out;
    if (f.tag_in) p.tag_in = f.tag_in;
    if (f.tag_expect) memcpy(p.tag_expect, f.tag_expect, 16);
    if (f.status) p.status = f.status;
    p.status_init = f.status_init;
}

// Long aligned messages under GCM_GHASH_TENSOR: three links of a chunk chain on the caller's stream.
//   1. AAD + the first T2_HEAD_BLOCKS payload blocks through the row kernel        -> state d_gt[0]
//   2. whole 128-block slices through gcm_tc2_kernel (AES warps + tensor-core GHASH) -> state d_gt[1], H^(blocks of 3) -> d_gt[2]
//   3. the rest and the length block through the row kernel, which finishes the tag / the compare
static bool tc2_takes(const gcm_ctx *c, const void *d_in, uint64_t len, const void *d_out)
{
    if ((((uintptr_t)d_in | (uintptr_t)d_out) & 15) != 0) return false;
    if (c->engine == GCM_GHASH_TENSOR) return len >= T2_MIN_BYTES;
    if (c->engine == GCM_GHASH_AUTO) return len >= (c->nr == 10 ? T2_AUTO_BYTES_128 : T2_AUTO_BYTES_256);
    return false;
}

// a link of the chain: header-sized, so the single-CTA latency kernel takes it when it can (no tickets drawn)
static cudaError_t launch_link(gcm_ctx *c, int mode, int blocks, const GcmParams &p, cudaStream_t s)
{
    const uint64_t n_ghash = (uint64_t)p.m.n_aad_blocks + (p.m.len + 15) / 16 + p.m.len_block;
    if (n_ghash <= SMALL_MAX_BLOCKS && p.stamps == nullptr) {
        c->ticket_next -= (unsigned)blocks;
        return launch_small(c->nr, mode, p, s);
    }
    return gcm_launch_fused(c, mode, blocks, p, s);
}

static int crypt_tc2_locked(gcm_ctx *c, int mode, const uint8_t iv[12], const void *d_aad, uint64_t aad_len, const void *d_in,
                            uint64_t len, void *d_out, const FinalOpts &fin, cudaStream_t s)
{
    const uint64_t head = 16ull * T2_HEAD_BLOCKS, nslices = (len / 16 - T2_HEAD_BLOCKS) / 128, bulk = nslices * 2048, tail = len - head - bulk;
    const uint8_t *in = (const uint8_t *)d_in;
    uint8_t *out = (uint8_t *)d_out;
    {   // the links only see their own stretch: the whole-message checks are made here
        const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
        if (a != b && a < b + len && b < a + len) return GCM_ERR_ARG;            // partial overlap
        if (aad_len >= (1ull << 61) || (aad_len + 15) / 16 > 0xFFFFFFFFull) return GCM_ERR_LEN;
    }
    GcmParams p;
    int blocks = 0;
    int rc = gcm_build_params(c, mode, iv, d_aad, aad_len, in, head, out, 0, false, len, aad_len, &p, &blocks);
    if (rc != GCM_OK) return rc;
    p.chain_out = c->d_gt + 0;
    cudaError_t e = launch_link(c, mode, blocks, p, s);
    secure_zero(&p, sizeof(p));
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    blocks = (int)(nslices < (uint64_t)c->grid ? nslices : (uint64_t)c->grid);
    c->ticket_next += (unsigned)blocks;
    e = launch_tc2(c->nr, mode, blocks, c->h_rk, c->h_te0, iv, T2_HEAD_BLOCKS + 2, in + head, out + head, nslices, c->d_bmat2, c->d_hx,
                   c->d_partials, c->d_counter, c->ticket_next - 1, c->d_gt + 0, c->d_gt + 1, (tail + 15) / 16 + 1, c->d_gt + 2,
                   reinterpret_cast<unsigned long long *>(c->d_gt + 4), s);
    if (e != cudaSuccess) { c->ticket_next -= (unsigned)blocks; return gcm_cuda_fail(e); }
    rc = gcm_build_params(c, mode, iv, nullptr, 0, in + head + bulk, tail, out + head + bulk, (uint32_t)(T2_HEAD_BLOCKS + 128 * nslices), true,
                          len, aad_len, &p, &blocks);
    if (rc != GCM_OK) return rc;
    p.chain_in = c->d_gt + 1;
    p.chain_pow = c->d_gt + 2;
    apply_final(p, fin);
    e = launch_link(c, mode, blocks, p, s);
    secure_zero(&p, sizeof(p));
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    return GCM_OK;
}

static int encrypt_async_locked(gcm_ctx *c, const uint8_t iv[12], const void *d_aad, uint64_t aad_len,
                                const void *d_pt, uint64_t len, void *d_ct, void *d_tag, void *stream)
{
    GcmParams p;
    int blocks = 0;
    if (!d_tag) return GCM_ERR_ARG;
    if (iv && tc2_takes(c, d_pt, len, d_ct) && len <= ((1ull << 36) - 32) && (!aad_len || d_aad)) {
        const FinalOpts fin = {(uint4 *)d_tag, nullptr, nullptr, nullptr, 0};
        return crypt_tc2_locked(c, MODE_ENCRYPT, iv, d_aad, aad_len, d_pt, len, d_ct, fin, (cudaStream_t)stream);
    }
    int rc = gcm_build_params(c, MODE_ENCRYPT, iv, d_aad, aad_len, d_pt, len, d_ct, 0, true, len, aad_len, &p, &blocks);
    if (rc != GCM_OK) return rc;
    p.tag_out = (uint4 *)d_tag;
    cudaError_t e = launch_auto(c, MODE_ENCRYPT, blocks, p, (cudaStream_t)stream);
    secure_zero(&p, sizeof(p));
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    return GCM_OK;
}

extern "C" int gcm_encrypt_async(gcm_ctx *c, const uint8_t iv[12], const void *d_aad, uint64_t aad_len,
                                 const void *d_pt, uint64_t len, void *d_ct, void *d_tag, void *stream)
{
    LOCK_CTX(c);
    return encrypt_async_locked(c, iv, d_aad, aad_len, d_pt, len, d_ct, d_tag, stream);
}

extern "C" int gcm_decrypt_verify_async(gcm_ctx *c, const uint8_t iv[12], const void *d_aad, uint64_t aad_len,
                                        const void *d_ct, uint64_t len, void *d_pt, const void *d_tag,
                                        void *d_status, void *stream)
{
    LOCK_CTX(c);
    GcmParams p;
    int blocks = 0;
    if (!d_tag || !d_status) return GCM_ERR_ARG;
    if (iv && tc2_takes(c, d_ct, len, d_pt) && len <= ((1ull << 36) - 32) && (!aad_len || d_aad)) {
        CU(cudaMemsetAsync(d_status, 0x7F, 4, (cudaStream_t)stream));       // reads "refused" (non-zero) until the last link has decided
        const FinalOpts fin = {nullptr, (const uint4 *)d_tag, nullptr, (int *)d_status, 1};
        int rc2 = crypt_tc2_locked(c, MODE_DECRYPT, iv, d_aad, aad_len, d_ct, len, d_pt, fin, (cudaStream_t)stream);
        if (rc2 != GCM_OK) return rc2;
        launch_wipe((uint8_t *)d_pt, len, (const int *)d_status, (cudaStream_t)stream);
        CU(cudaGetLastError());
        return GCM_OK;
    }
    int rc = gcm_build_params(c, MODE_DECRYPT, iv, d_aad, aad_len, d_ct, len, d_pt, 0, true, len, aad_len, &p, &blocks);
    if (rc != GCM_OK) return rc;
    p.tag_in = (const uint4 *)d_tag;
    p.status = (int *)d_status;
    p.status_init = 1;          // the verdict word reads "refused" until the finisher has written it (fail closed)
    cudaError_t e = launch_auto(c, MODE_DECRYPT, blocks, p, (cudaStream_t)stream);
    secure_zero(&p, sizeof(p));
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    // validation gate + payload suppression (L243), decided on the device
    launch_wipe((uint8_t *)d_pt, len, (const int *)d_status, (cudaStream_t)stream);
    CU(cudaGetLastError());
    return GCM_OK;
}

// GHASH only on the tensor cores: one launch of gcm_ghash_tc_kernel over [pad | AAD | C | length block].
static int ghash_tensor_locked(gcm_ctx *c, const void *d_aad, uint64_t aad_len, const void *d_c, uint64_t len,
                               void *d_out, cudaStream_t s)
{
    const uint64_t nchunks = ghash_tc_chunks(aad_len, len);
    const int blocks = (int)(nchunks < (uint64_t)c->grid ? nchunks : (uint64_t)c->grid);
    c->ticket_next += (unsigned)blocks;
    cudaError_t e = launch_ghash_tc(blocks, (const uint8_t *)d_aad, aad_len, (const uint8_t *)d_c, len, c->d_bmat2, c->d_ktab2, c->d_hx,
                                    c->d_partials, c->d_counter, c->ticket_next - 1, (uint4 *)d_out, s);
    if (e != cudaSuccess) { c->ticket_next -= (unsigned)blocks; return gcm_cuda_fail(e); }
    return GCM_OK;
}

extern "C" int gcm_ghash_async(gcm_ctx *c, const void *d_aad, uint64_t aad_len, const void *d_c, uint64_t len,
                               void *d_out, void *stream)
{
    LOCK_CTX(c);
    GcmParams p;
    int blocks = 0;
    if (!d_out) return GCM_ERR_ARG;
    if (c->engine != GCM_GHASH_TABLE && len >= (c->engine == GCM_GHASH_TENSOR ? GT_MIN_BYTES : GT_AUTO_BYTES) && d_c && ((uintptr_t)d_c & 15) == 0 &&
        len <= ((1ull << 36) - 32) && aad_len < (1ull << 32) && (!aad_len || d_aad))
        return ghash_tensor_locked(c, d_aad, aad_len, d_c, len, d_out, (cudaStream_t)stream);
    int rc = gcm_build_params(c, MODE_GHASH, nullptr, d_aad, aad_len, d_c, len, nullptr, 0, true, len, aad_len, &p, &blocks);
    if (rc != GCM_OK) return rc;
    p.tag_out = (uint4 *)d_out;
    cudaError_t e = gcm_launch_fused(c, MODE_GHASH, blocks, p, (cudaStream_t)stream);
    secure_zero(&p, sizeof(p));
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    return GCM_OK;
}

extern "C" int gcm_encrypt(gcm_ctx *c, const uint8_t iv[12], const void *d_aad, uint64_t aad_len,
                           const void *d_pt, uint64_t len, void *d_ct, uint8_t tag[16], void *stream)
{
    if (!tag) return GCM_ERR_ARG;
    LOCK_CTX(c);
    // the finishing thread stores the tag straight into mapped pinned host memory (unified addressing):
    // one posted PCIe write instead of a separate D2H copy on the latency path
    int rc = encrypt_async_locked(c, iv, d_aad, aad_len, d_pt, len, d_ct, c->h_pinned, stream);
    if (rc != GCM_OK) return rc;
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    memcpy(tag, c->h_pinned, 16);
    return GCM_OK;
}

extern "C" int gcm_decrypt_verify(gcm_ctx *c, const uint8_t iv[12], const void *d_aad, uint64_t aad_len,
                                  const void *d_ct, uint64_t len, void *d_pt, const uint8_t tag[16], void *stream)
{
    if (!tag) return GCM_ERR_ARG;
    LOCK_CTX(c);
    GcmParams p;
    int blocks = 0;
    // verdict written straight into mapped pinned host memory; it reads "refused" until the finisher says
    // otherwise, so a launch that never finishes cannot pass for an accepted message (fail closed)
    volatile int *verdict = (volatile int *)(c->h_pinned + 16);
    if (iv && tc2_takes(c, d_ct, len, d_pt) && len <= ((1ull << 36) - 32) && (!aad_len || d_aad)) {
        *verdict = GCM_STATUS_PENDING;
        const FinalOpts fin = {nullptr, nullptr, tag, (int *)(c->h_pinned + 16), 0};
        int rc2 = crypt_tc2_locked(c, MODE_DECRYPT, iv, d_aad, aad_len, d_ct, len, d_pt, fin, (cudaStream_t)stream);
        if (rc2 != GCM_OK) return rc2;
    } else {
    int rc = gcm_build_params(c, MODE_DECRYPT, iv, d_aad, aad_len, d_ct, len, d_pt, 0, true, len, aad_len, &p, &blocks);
    if (rc != GCM_OK) return rc;
    memcpy(p.tag_expect, tag, 16);      // expected tag travels by value; compared on the device
    *verdict = GCM_STATUS_PENDING;
    p.status = (int *)(c->h_pinned + 16);
    cudaError_t e = launch_auto(c, MODE_DECRYPT, blocks, p, (cudaStream_t)stream);
    secure_zero(&p, sizeof(p));
    if (e != cudaSuccess) return gcm_cuda_fail(e);
    }
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    if (*verdict != 0) {
        launch_wipe((uint8_t *)d_pt, len, nullptr, (cudaStream_t)stream);
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize((cudaStream_t)stream));
        return GCM_ERR_AUTH;
    }
    return GCM_OK;
}

// Diagnostics: the SM clock gcm_tc2_kernel ran at in the context's most recent chain (CTA 0's clock64 and %globaltimer
// at entry and exit, left in the context's scratch by the kernel itself).  Synchronises the device.
extern "C" int gcm_debug_tc2_clock(gcm_ctx *c, double *sm_mhz, double *kernel_ms)
{
    if (!c || !sm_mhz || !kernel_ms) return GCM_ERR_ARG;
    LOCK_CTX(c);
    unsigned long long v[4] = {0, 0, 0, 0};
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(v, c->d_gt + 4, sizeof(v), cudaMemcpyDeviceToHost));
    if (v[3] <= v[1] || v[2] <= v[0]) return GCM_ERR_ARG;          // no gcm_tc2 launch on this context yet
    *sm_mhz = (double)(v[2] - v[0]) / (double)(v[3] - v[1]) * 1e3;  // cycles per ns -> MHz
    *kernel_ms = (double)(v[3] - v[1]) * 1e-6;
    return GCM_OK;
}
