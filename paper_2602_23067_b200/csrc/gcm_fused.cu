// gcm_fused.cu -- the hot path: SURVEY.md 8(a) steps a3-a11 in ONE kernel.
//
//   AES-CTR keystream (a4, a5) -> XOR into the payload (a6) -> GHASH of the ciphertext while it is
//   still in registers (a7) -> per-thread / warp / CTA / cross-CTA combination with precomputed
//   powers of H (a8, a9) -> AAD + length block, E_K(J0), tag,
//   constant-time compare (a10, a11).
//
// What differs from the paper's kernels (prior art for Ampere/Ada/Hopper):
//   * one fused pass instead of an AES-CTR kernel followed by a GHASH kernel (the ciphertext never
//     crosses HBM twice);
//   * the "tree" is flattened.  The virtual block sequence [pad | AAD | payload | length block] is cut into
//     rows of 32 blocks; a warp owns a contiguous run of rows and lane l of the warp the l-th block of each.
//     Every lane therefore runs the SAME recurrence  Y <- Y.K xor X  with the one fixed multiplier
//     K = H^32 (independent of the launch geometry and of the message: the row loop of gcm_device.cuh), and is
//     corrected once by H^(1..32); the warp sums are weighted by H^(blocks behind the warp's run) in ONE
//     lane-parallel product by warp 0 (weights made by warp 0 while the tables arrive), and the CTA partials are
//     XORed by the last CTA to finish.  The sum is the paper's sum of X_i . H^(N-i+1); only the association
//     differs, and the field is exact, so the bits are identical;
//   * the multiply by the fixed K is an 8-bit Shoup table in shared memory (conflict-free by lane
//     rotation), AES rounds are T-tables replicated per lane (conflict-free, constant-time).  On
//     sm_100a the binding unit is the shared-memory pipe;
//   * counters of a lane's consecutive blocks differ by 32, so for 8 rows at a time only the low
//     counter byte changes: of rounds 1 and 2 only 1 + 4 table reads depend on it, the other 3 + 12
//     are cached per lane and refreshed every 8th row (in addition to the 12 round-1 reads of the
//     constant IV columns, done once per thread);
//   * Blackwell plumbing for the fixed cost per launch (the paper's FITS files are 17-577 MB, Table A.7,
//     where it matters): the 64 KB multiplier table arrives by one bulk copy (TMA 1-D, cp.async.bulk) completing on
//     an mbarrier while the threads expand the round table and warp 0 forms the position weights; the kernel is
//     launched with programmatic stream serialization, so its prologue overlaps the previous kernel's tail and
//     only griddepcontrol.wait orders it behind earlier work of the stream.
//
// Counter block of payload block g is IV || BE32(g + 2): a function of g only.
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_fused.cuh"

#include "gcm_device.cuh"

#include <atomic>
#include <stdlib.h>

#ifndef GHASH_PREFETCH_ROWS
#define GHASH_PREFETCH_ROWS 2       /* payload rows in flight per lane in GHASH-only mode (gcm_rows: DEPTH); measured on a
                                       B200, 4 GiB: 1 row 2032 GB/s, 2 rows 2111, 3 rows 2110, 4 rows 1590 */
#endif

#define STAMP(k)                                                                                   \
    do {                                                                                           \
        if (p.stamps != nullptr && threadIdx.x == 0) p.stamps[8 * blockIdx.x + (k)] = global_timer_ns(); \
    } while (0)

__device__ __forceinline__ uint4 warp_xor4(uint4 v)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        v.x ^= __shfl_xor_sync(0xFFFFFFFFu, v.x, o); v.y ^= __shfl_xor_sync(0xFFFFFFFFu, v.y, o);
        v.z ^= __shfl_xor_sync(0xFFFFFFFFu, v.z, o); v.w ^= __shfl_xor_sync(0xFFFFFFFFu, v.w, o);
    }
    return v;
}

// a8, first half, by warp 0 while the multiplier table is still on its way: D_w = H^(blocks behind the run of
// warp w of this CTA) for every warp of the CTA at once.  H^d for d < 2^36 is a product of four entries of the
// radix-512 digit table (PAPER.md L197 precomputes H^(2^k): 36 factors; radix 512 needs 4).  Lane j works for
// warp j >> 1 on digit pair j & 1, so the two product levels serve all (up to 16) warps in two generic products;
// messages below 2^18 / 2^9 blocks need one / none.  The tail run and runs without rows get H^0 = 1.
template <int NW>
__device__ __forceinline__ void cta_position_weights(const GcmParams &p, uint32_t lane, uint4 *wpow)
{
    const uint64_t E = p.m.vblocks;
    const uint32_t S = p.m.rows, w = lane >> 1, half = lane & 1;
    const uint64_t wg = (uint64_t)blockIdx.x * NW + w;
    const uint32_t r1 = (uint32_t)(((wg + 1) * S) / p.warps);
    const uint64_t d = (w < NW && r1 < S) ? E - 32ull * r1 : 0;
    const int levels = E < (1ull << HX_RADIX_BITS) ? 0 : (E < (1ull << (2 * HX_RADIX_BITS)) ? 1 : 2);
    const uint32_t k0 = 2 * half, k1 = 2 * half + 1, mask = (1u << HX_RADIX_BITS) - 1;
    uint4 f = __ldg(p.tab.hx + (k0 << HX_RADIX_BITS) + ((uint32_t)(d >> (HX_RADIX_BITS * k0)) & mask));
    if (levels >= 1) {
        const uint4 g = __ldg(p.tab.hx + (k1 << HX_RADIX_BITS) + ((uint32_t)(d >> (HX_RADIX_BITS * k1)) & mask));
        f = gf_mul_mem(f, g);
    }
    if (levels == 2) {
        uint4 g;
        g.x = __shfl_xor_sync(0xFFFFFFFFu, f.x, 1); g.y = __shfl_xor_sync(0xFFFFFFFFu, f.y, 1);
        g.z = __shfl_xor_sync(0xFFFFFFFFu, f.z, 1); g.w = __shfl_xor_sync(0xFFFFFFFFu, f.w, 1);
        f = gf_mul_mem(f, g);
    }
    if (half == 0 && w < NW) wpow[w] = f;
}

template <int NR, int MODE, int TPB>
__global__ void __launch_bounds__(TPB, 1)
gcm_fused_kernel(const __grid_constant__ GcmParams p)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    __shared__ uint4 s_ekj0;
    constexpr uint32_t NW = TPB / 32;
    const uint32_t t = threadIdx.x, lane = t & 31, lane4 = lane * 4;
    // broadcast from lane 0: tells the compiler the warp index (and the row loop) is warp-uniform,
    // so the shared-memory base stays in a uniform register and folds into every LDS address
    const uint32_t warp = __shfl_sync(0xFFFFFFFFu, t >> 5, 0);
    uint4 *red = reinterpret_cast<uint4 *>(sm + RED_OFF);
    uint4 *wpow = reinterpret_cast<uint4 *>(sm + WPOW_OFF);

    pdl_launch_dependents();            // the next launch of the stream may begin its own prologue
    STAMP(0);
    tables_begin<TPB, MODE != MODE_GHASH, true>(sm, p.tab, p.te0);

    // this warp's run of rows (geometry-agnostic: the result does not depend on it), balanced to +-1 row
    const uint32_t S = p.m.rows;
    const uint64_t wg = (uint64_t)blockIdx.x * NW + warp;
    // (the broadcasts keep the loop bounds in uniform registers: the 64-bit divisions hide from the compiler that
    // they are warp-uniform, and a row loop it takes for divergent cannot fold the shared-memory base into its LDS)
    const uint32_t r0 = __shfl_sync(0xFFFFFFFFu, (uint32_t)((wg * S) / p.warps), 0);
    const uint32_t r1 = __shfl_sync(0xFFFFFFFFu, (uint32_t)(((wg + 1) * S) / p.warps), 0);
    const bool has_rows = r0 < r1;
    // HBM latency of the run's first rows is paid now, under the table fill (and, in a train of launches, under
    // the previous kernel's tail), not after griddepcontrol.wait: prefetch them into L2
    {
        const uint32_t f0 = r0 > p.m.fast_lo ? r0 : p.m.fast_lo, f1 = r1 < p.m.fast_hi ? r1 : p.m.fast_hi;
#pragma unroll
        for (uint32_t k = 0; k < 2; k++)
            if (f0 + k < f1) prefetch_l2(p.m.in + 16 * (32ull * (f0 + k) + lane - p.m.base));
    }

    tables_wait(sm);
    STAMP(1);
    // a8, first half: only warp 0 reads the position weights (after the rows), so only warp 0 forms them, and the
    // other warps do not wait for it: under programmatic dependent launch this falls into the wait for the previous
    // kernel of the stream; in an isolated launch warp 0 starts its rows two generic products late
    if (warp == 0) cta_position_weights<NW>(p, lane, wpow);
    STAMP(7);

    const MulK8 mul(sm, lane);
    CtrConst cc = {0, 0, 0, 0};
    if (MODE != MODE_GHASH) {
        cc = ctr_const(p.rk, p.iv[0], p.iv[1], p.iv[2], sm, lane4);
        // a3: E_K(J0), J0 = IV || 0^31 || 1, by the last warp of every CTA while the others start their rows
        // (any CTA may turn out to be the finisher); it reaches the finishing thread through shared memory
        if (warp == NW - 1) {
            const CtrCache c1 = ctr_cache(p.rk, sm, lane4, cc, 1u);
            const uint4 ek = aes_ctr_block<NR>(p.rk, sm, lane4, cc, c1, 1u);
            if (lane == 0) s_ekj0 = ek;
        }
    }
    // Nothing above depends on earlier work of the stream (tables are per key and complete before gcm_init
    // returns); payload, AAD, partials, ticket and verdict do.
    pdl_wait();
    STAMP(2);
    if (MODE == MODE_DECRYPT && p.status_init && blockIdx.x == 0 && t == 0) *p.status = GCM_STATUS_PENDING;

    const ParamMsgView m{p.m};
    const uint4 Y = gcm_rows<NR, MODE, MODE == MODE_GHASH ? GHASH_PREFETCH_ROWS : 1>(m, p.rk, sm, lane, cc, r0, r1, mul);      // a4-a7
    STAMP(3);

    // a8, second half: one product per lane aligns it with the end of the warp's run, XOR over the warp;
    // warp 0 then weights the warp sums with their positions (one lane-parallel product) and XORs them
    uint4 part = make_uint4(0, 0, 0, 0);
    if (has_rows) {
        const uint32_t rem = r1 == S ? (uint32_t)(p.m.vblocks - 32ull * (S - 1)) : 32u;       // 1..32
        part = gf_mul_mem(Y, __ldg(p.tab.hpow + lane_exponent(rem, lane)));
    }
    part = warp_xor4(part);
    if (lane == 0) red[warp] = part;
    __syncthreads();
    STAMP(4);
    if (warp != 0) return;
    uint4 acc = make_uint4(0, 0, 0, 0), wgt = make_uint4(0, 0, 0, 0);
    if (lane < NW) { acc = red[lane]; wgt = wpow[lane]; }
    acc = warp_xor4(gf_mul_mem(acc, wgt));
    // a9: last-CTA-done combination of the CTA partials.  The ticket counter is never reset: the host hands
    // every launch the ticket value that ends it, so an aborted launch cannot leave a stale count behind.
    // One acquire-release atomic instead of two sequentially consistent fences (__threadfence is MEMBAR.SC + an L1
    // invalidation, twice on the tail of every launch): the release half publishes this CTA's partial, the acquire
    // half orders the finisher's reads (L2 reads, __ldcg) behind every other CTA's release.
    unsigned ticket = 0;
    if (lane == 0) {
        p.partials[blockIdx.x] = acc;
        asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(ticket) : "l"(p.counter) : "memory");
    }
    ticket = __shfl_sync(0xFFFFFFFFu, ticket, 0);
    STAMP(5);
    if (ticket != p.ticket_last) return;
    uint4 tot = make_uint4(0, 0, 0, 0);
    for (uint32_t j = lane; j < gridDim.x; j += 32) tot = xor4(tot, __ldcg(p.partials + j));
    tot = warp_xor4(tot);
    if (lane == 0) {
        if (p.chain_in != nullptr) tot = xor4(tot, gf_mul_mem(*p.chain_in, *p.chain_pow));
        if (p.chain_out != nullptr) {       // a middle chunk of a longer message: hand the state on
            *p.chain_out = tot;
        } else if (MODE == MODE_GHASH) {     // a10 is part of the rows: tot is GHASH_H(A, C)
            *p.tag_out = tot;
        } else {
            // a11: tag = E_K(J0) xor S; constant-time compare
            const uint4 tag = xor4(tot, s_ekj0);
            if (MODE == MODE_ENCRYPT) {
                *p.tag_out = tag;
            } else {
                uint4 expect = make_uint4(p.tag_expect[0], p.tag_expect[1], p.tag_expect[2], p.tag_expect[3]);
                if (p.tag_in != nullptr) expect = *p.tag_in;
                const uint32_t diff = (tag.x ^ expect.x) | (tag.y ^ expect.y) | (tag.z ^ expect.z) | (tag.w ^ expect.w);
                *p.status = diff != 0 ? 1 : 0;
            }
        }
    }
    STAMP(6);
}

// ---- host side ------------------------------------------------------------------------------------
// Programmatic stream serialization (on unless GCM_NO_PDL is set in the environment, for A/B measurements).
static bool pdl_enabled()
{
    static const bool on = getenv("GCM_NO_PDL") == nullptr;
    return on;
}

cudaError_t launch_with_pdl(const void *kern, dim3 grid, dim3 block, size_t smem, cudaStream_t s, void **args)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl_enabled() ? 1 : 0;
    return cudaLaunchKernelExC(&cfg, kern, args);
}

// The opt-in shared-memory size is a sticky per-function, per-device attribute: set once per (function, device).
cudaError_t ensure_smem_attr(const void *kern, std::atomic<bool> *configured, size_t bytes)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool tracked = dev >= 0 && dev < GCM_MAX_DEVICES;
    if (!tracked || !configured[dev].load(std::memory_order_acquire)) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        if (tracked) configured[dev].store(true, std::memory_order_release);      // setting it twice is harmless
    }
    return cudaSuccess;
}

template <int NR, int MODE, int TPB>
static cudaError_t launch_one(int blocks, const GcmParams &p, cudaStream_t s)
{
    static std::atomic<bool> configured[GCM_MAX_DEVICES];   // per instantiation and device
    const void *kern = (const void *)gcm_fused_kernel<NR, MODE, TPB>;
    cudaError_t e = ensure_smem_attr(kern, configured, FUSED_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    void *args[] = {(void *)&p};
    return launch_with_pdl(kern, dim3(blocks), dim3(TPB), FUSED_SMEM_BYTES, s, args);
}

template <int TPB>
static cudaError_t launch_tpb(int nr, int mode, int blocks, const GcmParams &p, cudaStream_t s)
{
    if (mode == MODE_GHASH) return launch_one<10, MODE_GHASH, TPB>(blocks, p, s);
    if (nr == 10) return mode == MODE_ENCRYPT ? launch_one<10, MODE_ENCRYPT, TPB>(blocks, p, s)
                                              : launch_one<10, MODE_DECRYPT, TPB>(blocks, p, s);
    return mode == MODE_ENCRYPT ? launch_one<14, MODE_ENCRYPT, TPB>(blocks, p, s)
                                : launch_one<14, MODE_DECRYPT, TPB>(blocks, p, s);
}

cudaError_t launch_fused(int nr, int mode, int threads, int blocks, const GcmParams &p, cudaStream_t s)
{
    if (threads == 256) return launch_tpb<256>(nr, mode, blocks, p, s);
    if (threads == 384) return launch_tpb<384>(nr, mode, blocks, p, s);
    return launch_tpb<512>(nr, mode, blocks, p, s);
}
