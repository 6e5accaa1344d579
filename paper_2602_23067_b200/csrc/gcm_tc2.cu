// gcm_tc2.cu -- AES-CTR + GHASH of a long stretch of whole, 16-byte-aligned payload blocks with the two halves of the
// path on different warps: the AES warps do nothing but AES (two rows at a time), the GHASH runs on the tensor cores
// from a shared-memory hand-over.  One link of the chunk chain of GcmParams (chain_in / chain_out): the row kernel
// (gcm_fused.cu) does the AAD and the first blocks in front of it and the ragged rest and the length block behind it.
//
// Why.  With the multiplier table gone from the shared-memory pipe (gcm_tc.cu) a warp has only
// its AES chain to issue from, and twelve warps of one dependent chain each leave that pipe a sixth idle; giving the
// same warps the tensor hand-over as well (bit expansion, tcgen05.st, barriers with a ring of two) made it worse.
// AES-CTR alone with two independent chains per lane runs at 705 GB/s on 12 warps (0.94 of the AES table-read bound).
// So here:
//   * 12 AES warps.  The CTA's run is cut into slices of 128 consecutive blocks (4 rows of 32); slice t belongs to AES
//     warp t mod 12, which loads it, runs rows (0, 1) and (2, 3) as pairs (one ctr_cache per slice: the stretch starts
//     at a counter that is 0 mod 256, so a slice never straddles an 8-row counter group), stores the output, and leaves
//     the GHASH input (ciphertext) in a 2 KB stage of shared memory: four STS.128 and one mbarrier arrival per slice.
//   * 4 GHASH warps (one per TMEM lane quarter) take the stages in order: row q of the slice, LDS.128, bit expansion
//     (gcm_tc.cu), tcgen05.st into a ring of 12 slices in TMEM.  Block 128 t + j of the run is row j of slice t, so the
//     slice weights are powers of K = H^128 (the matrices of gcm_ghash_tc.cu).
//   * 1 warp issues the MMAs.  A chunk is L = 7 slices and the running value: acc = sum X_s . K^(l-1-s) + Y . K^l.
//     Two accumulators alternate; the GHASH warps read chunk c-1 back (parity of the counts) while chunk c's slices are
//     multiplied, and hand Y in as chunk c's LAST slice.
// Shared memory: 128 KB AES tables + 8 matrices of 8 KB + 16 stages of 2 KB.  TMEM: 2 x 128 accumulator columns, 32 of
// scale factors, 2 x 16 for Y, 12 x 16 ring.  17 warps (96 registers each).
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_fused.cuh"
#include "gcm_tc.cuh"
#include "gcm_api_internal.h"

#include "gcm_device.cuh"

#include <atomic>
#include <string.h>

#define T2_AES       12
#define T2_THREADS   (32 * (T2_AES + 4 + 1))
#define T2_L         7                               /* slices per chunk */
#define T2_STAGES    16
#define T2_RING      12
#define T2_COL_SF    256
#define T2_COL_Y     288
#define T2_COL_RING  320
#define T2_BMAT_OFF  AES_TAB_BYTES
#define T2_STAGE_OFF (T2_BMAT_OFF + (T2_L + 1) * TC_BMAT_BYTES)
#define T2_RED_OFF   (T2_STAGE_OFF + T2_STAGES * 2048)
#define T2_BAR_OFF   (T2_RED_OFF + 128)              /* tabbar, sfull[16], sempty[16], tfull[12], tempty[12], yfull[2], accfull[2] */
#define T2_SMEM_BYTES (T2_BAR_OFF + 64 * 8 + 16)
#define T2_IDESC ((1u << 7) | (1u << 10) | (16u << 17) | (1u << 23) | (8u << 24))
static_assert(T2_L + 1 <= GT_L, "the matrices of H^(128 e), e <= T2_L, come from the GHASH-only kernel's set");

struct Tc2Params {
    uint32_t rk[60];
    uint32_t te0[256];
    uint32_t iv[3];
    uint32_t ctr0;              // counter of the stretch's first block: 0 mod 256
    const uint8_t *in;
    uint8_t *out;
    uint64_t nslices;           // 128 blocks each
    const uint4 *bmat2;
    const uint4 *hx;
    uint4    *partials;
    unsigned *counter;
    unsigned  ticket_last;
    const uint4 *chain_in;      // GHASH state in front of the stretch, or NULL
    uint4    *chain_out;        // state behind it
    uint64_t  exp_next;         // H^exp_next goes to pow_out: chain_pow of the launch that follows
    uint4    *pow_out;
    unsigned long long *clk;    // diagnostics, or NULL: CTA 0 leaves {clock64, %globaltimer} of its entry and exit here (4 words)
};

__device__ __forceinline__ void t2_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void t2_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void t2_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// The helper warps spend most of their time waiting; a try_wait that comes back every few dozen cycles costs issue
// slots and MIO bandwidth the AES warps need (105 SYNCS per warp-row were measured), so the wait carries a suspend-time
// hint: the hardware parks the warp until the phase completes or the hint runs out.
__device__ __forceinline__ void t2_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
    } while (!done);
}
__device__ __forceinline__ bool t2_elect()
{
    uint32_t pred;
    asm volatile("{ .reg .pred p; elect.sync _|p, 0xFFFFFFFF; selp.u32 %0, 1, 0, p; }" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void t2_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void t2_mma(uint32_t d, uint32_t a, uint64_t b, uint32_t sf, uint32_t accumulate)
{
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %5, 0;\n"
                 "tcgen05.mma.cta_group::1.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%4], [%4], p;\n}"
                 ::"r"(d), "r"(a), "l"(b), "r"(T2_IDESC), "r"(sf), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void t2_st16(uint32_t taddr, uint4 x)
{
    uint32_t v[16];
    const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
    for (int c = 0; c < 4; c++) {
        v[4 * c + 0] = w[c] & 0x11111111u;                      // bits 0, 4, ..: e2m1 0.5
        v[4 * c + 1] = w[c] & 0x22222222u;                      // bits 1, 5, ..: 1.0
        v[4 * c + 2] = w[c] & 0x44444444u;                      // bits 2, 6, ..: 2.0
        v[4 * c + 3] = (w[c] >> 1) & 0x44444444u;               // bits 3, 7, ..: 2.0
    }
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                   "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t t2_ld_parity32(uint32_t taddr)
{
    uint32_t r[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                   "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    uint32_t w = 0;
#pragma unroll
    for (int base = 0; base < 32; base += 11) {
        uint32_t acc = 0;
#pragma unroll
        for (int i = 0; i < 11; i++)
            if (base + i < 32) {
                const float t = __fmaf_rn(__uint_as_float(r[base + i]), (float)(1u << i), 8388608.0f);
                acc |= __float_as_uint(t) & (1u << i);
            }
        w |= acc << base;
    }
    return w;
}
__device__ __forceinline__ uint4 t2_warp_xor4(uint4 v)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        v.x ^= __shfl_xor_sync(0xFFFFFFFFu, v.x, o); v.y ^= __shfl_xor_sync(0xFFFFFFFFu, v.y, o);
        v.z ^= __shfl_xor_sync(0xFFFFFFFFu, v.z, o); v.w ^= __shfl_xor_sync(0xFFFFFFFFu, v.w, o);
    }
    return v;
}
__device__ __forceinline__ uint4 t2_pow(const uint4 *hx, uint64_t d)           // H^d from the radix-512 digit tables
{
    const uint32_t mask = (1u << HX_RADIX_BITS) - 1;
    uint4 r = __ldg(hx + ((uint32_t)d & mask));
    for (uint32_t dig = 1; dig < HX_DIGITS; dig++) {
        const uint32_t j = (uint32_t)(d >> (HX_RADIX_BITS * dig)) & mask;
        if (j) r = gf_mul_mem(r, __ldg(hx + (dig << HX_RADIX_BITS) + j));
    }
    return r;
}

template <int NR, int MODE>
__global__ void __launch_bounds__(T2_THREADS, 1)
gcm_tc2_kernel(const __grid_constant__ Tc2Params p)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    const uint32_t t = threadIdx.x, lane = t & 31, lane4 = lane * 4;
    const uint32_t warp = __shfl_sync(0xFFFFFFFFu, t >> 5, 0);
    uint4 *red = reinterpret_cast<uint4 *>(sm + T2_RED_OFF);
    const uint32_t bars = smem_u32(sm + T2_BAR_OFF);
    const uint32_t tabbar = bars, sfull = bars + 8, sempty = sfull + 8 * T2_STAGES, tfull = sempty + 8 * T2_STAGES,
                   tempty = tfull + 8 * T2_RING, yfull = tempty + 8 * T2_RING, accfull = yfull + 16;
    uint32_t *tslot = reinterpret_cast<uint32_t *>(sm + T2_BAR_OFF + 64 * 8);
    const uint32_t stage0 = smem_u32(sm + T2_STAGE_OFF);

    pdl_launch_dependents();
    const uint64_t s0 = (p.nslices * blockIdx.x) / gridDim.x, s1 = (p.nslices * (blockIdx.x + 1)) / gridDim.x;
    const uint32_t T = (uint32_t)(s1 - s0);
    if (warp == T2_AES + 4) {
        if (lane == 0) {
            // SM clock this kernel really runs at (the tensor pipe lowers it below what nvidia-smi reports): cycles and
            // nanoseconds of CTA 0's life, stored at once so that no register is held across the AES warps' loop
            if (blockIdx.x == 0 && p.clk != nullptr) { p.clk[0] = (unsigned long long)clock64(); p.clk[1] = global_timer_ns(); }
            uint64_t *b = reinterpret_cast<uint64_t *>(sm + T2_BAR_OFF);
            mbar_init(b + 0, 1);
            for (int i = 0; i < T2_STAGES; i++) { mbar_init(b + 1 + i, 1); mbar_init(b + 1 + T2_STAGES + i, 4); }
            for (int i = 0; i < T2_RING; i++) { mbar_init(b + 1 + 2 * T2_STAGES + i, 4); mbar_init(b + 1 + 2 * T2_STAGES + T2_RING + i, 1); }
            for (int i = 0; i < 2; i++) { mbar_init(b + 1 + 2 * T2_STAGES + 2 * T2_RING + i, 4); mbar_init(b + 3 + 2 * T2_STAGES + 2 * T2_RING + i, 1); }
            mbar_expect_tx(b + 0, (T2_L + 1) * TC_BMAT_BYTES);
            for (int e = 0; e <= T2_L; e++)
                bulk_copy_g2s(sm + T2_BMAT_OFF + e * TC_BMAT_BYTES, reinterpret_cast<const uint8_t *>(p.bmat2) + e * TC_BMAT_BYTES, TC_BMAT_BYTES, b + 0);
        }
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tslot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    } else if (warp < T2_AES) {
        fill_aes_tables<32 * T2_AES>(sm, p.te0, t);
    }
    t2_fence_before();
    __syncthreads();
    t2_fence_after();
    const uint32_t tb = __shfl_sync(0xFFFFFFFFu, *tslot, 0);
    if (warp >= T2_AES && warp < T2_AES + 4) {           // scale factors: every byte 2^0 (UE8M0 127)
        const uint32_t one = 0x7F7F7F7Fu, a = tb + ((32u * (warp - T2_AES)) << 16) + T2_COL_SF;
#pragma unroll
        for (int c = 0; c < 32; c += 8)
            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(a + c), "r"(one) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    t2_fence_before();
    __syncthreads();
    t2_fence_after();

    if (warp < T2_AES) {
        // ---- AES warps: slices warp, warp + 12, ...; rows (0, 1) and (2, 3) of a slice side by side -------------------
        const CtrConst cc = ctr_const(p.rk, p.iv[0], p.iv[1], p.iv[2], sm, lane4);
        pdl_wait();
        uint32_t tt = warp;
        const uint64_t first = 16 * (128 * (s0 + tt) + lane);
        const uint8_t *src = p.in + first;
        uint8_t *dst = p.out + first;
        uint32_t ctr = p.ctr0 + (uint32_t)(128 * (s0 + tt)) + lane;
        uint4 x0 = make_uint4(0, 0, 0, 0), x1 = x0, x2 = x0, x3 = x0;
        if (tt < T) { x0 = ld16_stream(src); x1 = ld16_stream(src + 512); x2 = ld16_stream(src + 1024); x3 = ld16_stream(src + 1536); }
        for (; tt < T; tt += T2_AES) {
            uint4 n0 = make_uint4(0, 0, 0, 0), n1 = n0, n2 = n0, n3 = n0;
            if (tt + T2_AES < T) {                                      // this warp's next slice
                const uint8_t *nx = src + 2048 * T2_AES;
                n0 = ld16_stream(nx); n1 = ld16_stream(nx + 512); n2 = ld16_stream(nx + 1024); n3 = ld16_stream(nx + 1536);
            }
            const CtrCache cu = ctr_cache(p.rk, sm, lane4, cc, ctr);    // the slice's four counters share their upper 24 bits
            const uint32_t st = stage0 + 2048 * (tt & (T2_STAGES - 1)) + 16 * lane;
            {
                const uint4 ka = aes_ctr_block<NR>(p.rk, sm, lane4, cc, cu, ctr);
                const uint4 kb = aes_ctr_block<NR>(p.rk, sm, lane4, cc, cu, ctr + 32);
                const uint4 ya = xor4(x0, ka), yb = xor4(x1, kb);
                st16_stream(dst, ya);
                st16_stream(dst + 512, yb);
                t2_wait(sempty + 8 * (tt & (T2_STAGES - 1)), ((tt / T2_STAGES) & 1) ^ 1);     // the stage's previous slice has been taken
                const uint4 ga = MODE == MODE_ENCRYPT ? ya : x0, gb = MODE == MODE_ENCRYPT ? yb : x1;
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(st), "r"(ga.x), "r"(ga.y), "r"(ga.z), "r"(ga.w) : "memory");
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(st + 512), "r"(gb.x), "r"(gb.y), "r"(gb.z), "r"(gb.w) : "memory");
            }
            {
                const uint4 ka = aes_ctr_block<NR>(p.rk, sm, lane4, cc, cu, ctr + 64);
                const uint4 kb = aes_ctr_block<NR>(p.rk, sm, lane4, cc, cu, ctr + 96);
                const uint4 ya = xor4(x2, ka), yb = xor4(x3, kb);
                st16_stream(dst + 1024, ya);
                st16_stream(dst + 1536, yb);
                const uint4 ga = MODE == MODE_ENCRYPT ? ya : x2, gb = MODE == MODE_ENCRYPT ? yb : x3;
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(st + 1024), "r"(ga.x), "r"(ga.y), "r"(ga.z), "r"(ga.w) : "memory");
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(st + 1536), "r"(gb.x), "r"(gb.y), "r"(gb.z), "r"(gb.w) : "memory");
            }
            __syncwarp();
            if (lane == 0) t2_arrive(sfull + 8 * (tt & (T2_STAGES - 1)));
            x0 = n0; x1 = n1; x2 = n2; x3 = n3;
            src += 2048 * T2_AES; dst += 2048 * T2_AES; ctr += 128 * T2_AES;
        }
    } else if (warp < T2_AES + 4) {
        // ---- GHASH warps: row q of every slice, in order; chunk results back in as the next chunk's last slice ---------
        const uint32_t q = warp - T2_AES;
        const uint32_t lanebase = tb + ((32u * q) << 16);
        const uint32_t mine = stage0 + 512 * q + 16 * lane;
        uint4 Y = make_uint4(0, 0, 0, 0);
        // the three powers of H the finish needs, worked out now, while the first slices are still being encrypted: the
        // weight of this CTA's run, and (used by whichever CTA draws the last ticket) those of the chained state
        if (lane == 0 && q < 3) {
            const uint64_t e = q == 0 ? (p.nslices - s1) * 128 : q == 1 ? p.nslices * 128 : p.exp_next;
            red[4 + q] = t2_pow(p.hx, e);
        }
        uint32_t c = 0, s_in = 0, left = T, ell = left < T2_L ? left : T2_L, slot = 0, ph = 1;
        for (uint32_t tt = 0; tt < T; tt++) {
            const uint32_t sg = tt & (T2_STAGES - 1);
            t2_wait(sfull + 8 * sg, (tt / T2_STAGES) & 1);
            uint4 x;
            asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(x.x), "=r"(x.y), "=r"(x.z), "=r"(x.w) : "r"(mine + 2048 * sg) : "memory");
            t2_wait(tempty + 8 * slot, ph);
            t2_fence_after();
            t2_st16(lanebase + T2_COL_RING + 16 * slot, x);             // (the load above has completed: its data was used)
            t2_fence_before();
            __syncwarp();
            if (lane == 0) { t2_arrive(sempty + 8 * sg); t2_arrive(tfull + 8 * slot); }
            if (++slot == T2_RING) { slot = 0; ph ^= 1; }
            if (++s_in == ell) {
                if (c > 0) {                                            // chunk c - 1 back, in again as chunk c's last slice
                    const uint32_t b = (c - 1) & 1;
                    t2_wait(accfull + 8 * b, ((c - 1) >> 1) & 1);
                    t2_fence_after();
                    Y.x = t2_ld_parity32(lanebase + 128 * b + 0);
                    Y.y = t2_ld_parity32(lanebase + 128 * b + 32);
                    Y.z = t2_ld_parity32(lanebase + 128 * b + 64);
                    Y.w = t2_ld_parity32(lanebase + 128 * b + 96);
                    t2_st16(lanebase + T2_COL_Y + 16 * (c & 1), Y);
                    t2_fence_before();
                    __syncwarp();
                    if (lane == 0) t2_arrive(yfull + 8 * (c & 1));
                }
                c++; s_in = 0; left -= ell;
                ell = left < T2_L ? left : T2_L;
            }
        }
        uint4 part = make_uint4(0, 0, 0, 0);
        if (T) {
            const uint32_t b = (c - 1) & 1;
            t2_wait(accfull + 8 * b, ((c - 1) >> 1) & 1);
            t2_fence_after();
            Y.x = t2_ld_parity32(lanebase + 128 * b + 0);
            Y.y = t2_ld_parity32(lanebase + 128 * b + 32);
            Y.z = t2_ld_parity32(lanebase + 128 * b + 64);
            Y.w = t2_ld_parity32(lanebase + 128 * b + 96);
            part = gf_mul_mem(Y, __ldg(p.hx + (128 - (32 * q + lane))));   // row j ends 128 - j blocks before the run does
        }
        part = t2_warp_xor4(part);
        if (lane == 0) red[q] = part;
    } else {
        // ---- the issuing warp (every lane walks the loop; one elected lane issues) -------------------------------------
        t2_wait(tabbar, 0);
        const uint32_t sf = tb + T2_COL_SF;
        const uint64_t d0 = (uint64_t)((smem_u32(sm + T2_BMAT_OFF) >> 4) & 0x3FFF) | ((uint64_t)(2048 >> 4) << 16) | ((uint64_t)(128 >> 4) << 32) | (1ull << 46);
        uint32_t left = T, slot = 0, ph = 0;
        for (uint32_t c = 0; left; c++) {
            const uint32_t ell = left < T2_L ? left : T2_L, b = c & 1, d = tb + 128 * b;
            left -= ell;
            for (uint32_t s = 0; s < ell; s++) {
                t2_wait(tfull + 8 * slot, ph);
                t2_fence_after();
                const uint64_t dm = d0 + (uint64_t)((ell - 1 - s) * (TC_BMAT_BYTES >> 4));      // matrix of K^(ell-1-s)
                if (t2_elect()) {
                    t2_mma(d, tb + T2_COL_RING + 16 * slot, dm, sf, s);
                    t2_mma(d, tb + T2_COL_RING + 16 * slot + 8, dm + 256, sf, 1);
                    t2_commit(tempty + 8 * slot);
                }
                __syncwarp();
                if (++slot == T2_RING) { slot = 0; ph ^= 1; }
            }
            if (c > 0) {
                t2_wait(yfull + 8 * b, ((c - 1) >> 1) & 1);            // chunks 1, 3, .. use yfull[1]; 2, 4, .. yfull[0]
                t2_fence_after();
                const uint64_t dm = d0 + (uint64_t)(ell * (TC_BMAT_BYTES >> 4));                  // Y . K^ell
                if (t2_elect()) {
                    t2_mma(d, tb + T2_COL_Y + 16 * b, dm, sf, 1);
                    t2_mma(d, tb + T2_COL_Y + 16 * b + 8, dm + 256, sf, 1);
                }
                __syncwarp();
            }
            if (t2_elect()) t2_commit(accfull + 8 * b);
            __syncwarp();
        }
    }
    t2_fence_before();
    __syncthreads();
    t2_fence_after();
    if (warp != T2_AES + 4) return;
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tb) : "memory");
    unsigned ticket = 0;
    if (lane == 0) {
        uint4 acc = xor4(xor4(red[0], red[1]), xor4(red[2], red[3]));
        const uint64_t behind = (p.nslices - s1) * 128;
        if (behind && T) acc = gf_mul_mem(acc, red[4]);
        pdl_wait();
        if (blockIdx.x == 0 && p.clk != nullptr) { p.clk[2] = (unsigned long long)clock64(); p.clk[3] = global_timer_ns(); }
        p.partials[blockIdx.x] = acc;
        asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(ticket) : "l"(p.counter) : "memory");
    }
    ticket = __shfl_sync(0xFFFFFFFFu, ticket, 0);
    if (ticket != p.ticket_last) return;
    uint4 tot = make_uint4(0, 0, 0, 0);
    for (uint32_t j = lane; j < gridDim.x; j += 32) tot = xor4(tot, __ldcg(p.partials + j));
    tot = t2_warp_xor4(tot);
    if (lane == 0) {
        if (p.chain_in != nullptr) tot = xor4(tot, gf_mul_mem(*p.chain_in, red[5]));
        *p.chain_out = tot;
        if (p.pow_out != nullptr) *p.pow_out = red[6];
    }
}

template <int NR, int MODE>
static cudaError_t tc2_launch_one(int blocks, const Tc2Params &p, cudaStream_t s)
{
    static std::atomic<bool> configured[GCM_MAX_DEVICES];
    const void *kern = (const void *)gcm_tc2_kernel<NR, MODE>;
    cudaError_t e = ensure_smem_attr(kern, configured, T2_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    void *args[] = {(void *)&p};
    return launch_with_pdl(kern, dim3(blocks), dim3(T2_THREADS), T2_SMEM_BYTES, s, args);
}

// nr 10 / 14; mode MODE_ENCRYPT / MODE_DECRYPT; nslices * 128 whole blocks from `in` to `out` (both 16-byte aligned),
// the first of them with counter ctr0 (0 mod 256); GHASH state chained as in GcmParams.
cudaError_t launch_tc2(int nr, int mode, int blocks, const uint32_t *rk, const uint32_t *te0, const uint8_t *iv, uint32_t ctr0,
                       const uint8_t *in, uint8_t *out, uint64_t nslices, const uint4 *bmat2, const uint4 *hx, uint4 *partials,
                       unsigned *counter, unsigned ticket_last, const uint4 *chain_in, uint4 *chain_out, uint64_t exp_next,
                       uint4 *pow_out, unsigned long long *clk, cudaStream_t s)
{
    Tc2Params p;
    memset(&p, 0, sizeof(p));
    memcpy(p.rk, rk, sizeof(p.rk));
    memcpy(p.te0, te0, sizeof(p.te0));
    memcpy(p.iv, iv, 12);
    p.ctr0 = ctr0; p.in = in; p.out = out; p.nslices = nslices; p.bmat2 = bmat2; p.hx = hx;
    p.partials = partials; p.counter = counter; p.ticket_last = ticket_last;
    p.chain_in = chain_in; p.chain_out = chain_out; p.exp_next = exp_next; p.pow_out = pow_out; p.clk = clk;
    cudaError_t e;
    if (nr == 10) e = mode == MODE_ENCRYPT ? tc2_launch_one<10, MODE_ENCRYPT>(blocks, p, s) : tc2_launch_one<10, MODE_DECRYPT>(blocks, p, s);
    else e = mode == MODE_ENCRYPT ? tc2_launch_one<14, MODE_ENCRYPT>(blocks, p, s) : tc2_launch_one<14, MODE_DECRYPT>(blocks, p, s);
    secure_zero(&p, sizeof(p));
    return e;
}
