// gcm_ghash_tc.cu -- GHASH of a long, 16-byte-aligned stretch of ciphertext on the tensor cores (tcgen05 / TMEM).
//
// The paper's only like-for-like kernel figure is GHASH alone (Table 5 "GHashKernelOnly");
// SURVEY.md 8(f)-1.  Eq. 1 (L191) regrouped as in gcm_tc.cu -- the multiply by a fixed field element is a 128 x 128 bit
// matrix, XOR is the parity of a count, tcgen05.mma kind::mxf4 with e2m1 operands 0 / 0.5 / 1 / 2 counts exactly in
// fp32 -- but laid out for a kernel that has nothing else to do:
//
//   * ONE tile per CTA.  The CTA's run of blocks is cut into slices of 128 consecutive blocks; block 128 t + j of the
//     run is row j (TMEM lane j) of slice t.  A load warp brings the slices into shared memory (one bulk copy of 2 KB each, 16 in flight); twelve producer warps take their 16 bytes,
//     expand the bits to nibbles (five ALU instructions per word) and store their 32 rows of a slice straight into
//     TMEM (tcgen05.st); slice t belongs to the four warps with (warp >> 2) == t % 3, one per lane quarter.
//   * A chunk is 16 slices: row j of the accumulator becomes  Z_j = sum_t X_(128 t + j) . K^(15 - t),  K = H^128, by
//     32 MMAs with the bit matrices of K^15 .. K^0 as the B operand (128 KB of shared memory, loaded once).
//     One lane of one warp issues them; the accumulator is double-buffered (2 x 128 TMEM columns), the A ring holds
//     twelve slices, so producers, tensor core and read-back never wait for one another in steady state.
//   * Four read-back warps take the parity of the counts (tcgen05.ld, one FFMA + one LOP3 per count) and fold the
//     chunk into the row's running value  Y_j <- Y_j . K^16 xor Z_j  with the 8-bit table multiply of the fused
//     kernel (ghash_mul_k, table of H^2048): one table multiply per 16 blocks instead of one per block.
//   * End of the run: Y_j . H^(128 - j), XOR over the rows, times H^(blocks of the stretch behind the run), partial
//     to global memory, last-CTA-done as in gcm_fused.cu; the finisher adds the state handed in (chain_in . H^N) and
//     writes GHASH_H(A, C).  The kernel covers the WHOLE virtual sequence [pad | AAD | C | length block] (pad = leading
//     zero blocks up to a whole number of chunks): the few slices at both ends that are not whole blocks of C are put
//     together by the load warp with ordinary loads, all others arrive by bulk copy.  One launch per call.
//
// Bound: 32 MMAs of 64 cycles per 2048 blocks = one block per SM-cycle on the tensor pipe (4.65 TB/s at 1965 MHz),
// against two cycles per block on the shared-memory pipe for the table multiply and 0.73 for HBM (1 B/B at 6.5 TB/s).
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_fused.cuh"
#include "gcm_tc.cuh"

#include "gcm_device.cuh"

#include <atomic>
#include <string.h>

#define GT_PRODUCERS  12                             /* 17 warps are allotted registers as 20: 96 per thread */
#define GT_THREADS    (32 * (GT_PRODUCERS + 4 + 2))     /* + 4 read-back warps, the MMA warp, the load warp */
#define GT_STAGES     16                             /* 2 KB slices of the message in flight in shared memory (bulk copies) */
#define GT_RING       12                             /* A slices in TMEM */
#define GT_COL_SF     256
#define GT_COL_RING   288
#define GT_BMAT_OFF   0                              /* 16 x 8 KB; ktab2 follows at KTAB_OFF = 128 KB (ghash_mul_k reads it there) */
#define GT_STAGE_OFF  (KTAB_OFF + KTAB_BYTES)        /* GT_STAGES x 2 KB */
#define GT_RED_OFF    (GT_STAGE_OFF + GT_STAGES * 2048)
#define GT_BAR_OFF    (GT_RED_OFF + 64)              /* tabbar, full[12], empty[12], accfull[2], accempty[2], sfull[16], sempty[16] */
#define GT_SMEM_BYTES (GT_BAR_OFF + 64 * 8 + 16)
#define GT_IDESC ((1u << 7) | (1u << 10) | (16u << 17) | (1u << 23) | (8u << 24))
static_assert(GT_RING % (GT_PRODUCERS / 4) == 0, "a warp's slices keep their ring phase");
static_assert(GT_STAGES % (GT_PRODUCERS / 4) != 0 || true, "");
static_assert(GT_RING % 4 == 0 && GT_L % 4 == 0, "the issue loop takes four slices per trip");
static_assert(GT_BMAT_TOTAL == KTAB_OFF, "the matrices fill the 128 KB in front of the multiplier table");

// The kernel hashes the virtual block sequence  [pad zero blocks | AAD blocks | C blocks | length block]  of
// nchunks * GT_CHUNK_BLOCKS blocks: pad (leading zero blocks are free in GHASH) rounds it up to whole chunks, so the
// length block is the last block of the last chunk and nothing is left for another launch.
struct GhashTcParams {
    const uint8_t *in;          // C, 16-byte aligned
    const uint8_t *aad;
    uint64_t len, aad_len;      // bytes
    uint64_t pad, base;         // leading zero blocks; virtual index of C block 0 = pad + AAD blocks
    uint64_t nchunks;
    const uint4 *bmat2;         // GT_BMAT_TOTAL
    const uint4 *ktab2;         // KTAB_BYTES: Shoup table of H^(128 * GT_L)
    const uint4 *hx;
    uint4    *partials;
    unsigned *counter;
    unsigned  ticket_last;
    const uint4 *chain_in;      // GHASH state in front of the stretch, or NULL
    uint4    *chain_out;        // state behind it
    uint64_t  exp_next;         // H^exp_next is stored to pow_out (chain_pow of the launch that follows)
    uint4    *pow_out;
};

__device__ __forceinline__ void gt_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void gt_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void gt_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool gt_elect()
{
    uint32_t pred;
    asm volatile("{ .reg .pred p; elect.sync _|p, 0xFFFFFFFF; selp.u32 %0, 1, 0, p; }" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void mbar_wait_addr(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void gt_commit_addr(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void gt_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ uint64_t gt_smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | (1ull << 46);
}
__device__ __forceinline__ void gt_mma(uint32_t d, uint32_t a, uint64_t b, uint32_t sf, uint32_t accumulate)
{
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %5, 0;\n"
                 "tcgen05.mma.cta_group::1.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%4], [%4], p;\n}"
                 ::"r"(d), "r"(a), "l"(b), "r"(GT_IDESC), "r"(sf), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void gt_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                   "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
// 32 counts (fp32, <= 2048) -> 32 parity bits: c . 2^i + 2^23 has bit 0 of c at mantissa bit i
__device__ __forceinline__ uint32_t gt_parity32(const uint32_t (&r)[32])
{
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
__device__ __forceinline__ uint4 gt_warp_xor4(uint4 v)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        v.x ^= __shfl_xor_sync(0xFFFFFFFFu, v.x, o); v.y ^= __shfl_xor_sync(0xFFFFFFFFu, v.y, o);
        v.z ^= __shfl_xor_sync(0xFFFFFFFFu, v.z, o); v.w ^= __shfl_xor_sync(0xFFFFFFFFu, v.w, o);
    }
    return v;
}
// H^d, d < 2^36, from the radix-512 digit tables (one thread)
__device__ __forceinline__ uint4 gt_pow(const uint4 *hx, uint64_t d)
{
    const uint32_t mask = (1u << HX_RADIX_BITS) - 1;
    uint4 r = __ldg(hx + ((uint32_t)d & mask));
    for (uint32_t dig = 1; dig < HX_DIGITS; dig++) {
        const uint32_t j = (uint32_t)(d >> (HX_RADIX_BITS * dig)) & mask;
        if (j) r = gf_mul_mem(r, __ldg(hx + (dig << HX_RADIX_BITS) + j));
    }
    return r;
}

__global__ void __launch_bounds__(GT_THREADS, 1)
gcm_ghash_tc_kernel(const __grid_constant__ GhashTcParams p)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    const uint32_t t = threadIdx.x, lane = t & 31;
    const uint32_t warp = __shfl_sync(0xFFFFFFFFu, t >> 5, 0);
    uint4 *red = reinterpret_cast<uint4 *>(sm + GT_RED_OFF);
    uint64_t *bars = reinterpret_cast<uint64_t *>(sm + GT_BAR_OFF);
    uint64_t *full = bars + 1, *empty = bars + 1 + GT_RING, *accfull = bars + 1 + 2 * GT_RING, *accempty = accfull + 2;
    uint64_t *sfull = accempty + 2, *sempty = sfull + GT_STAGES;
    uint32_t *tslot = reinterpret_cast<uint32_t *>(sm + GT_BAR_OFF + 64 * 8);

    pdl_launch_dependents();
    // this CTA's chunks [c0, c1) of the stretch
    const uint64_t c0 = (p.nchunks * blockIdx.x) / gridDim.x, c1 = (p.nchunks * (blockIdx.x + 1)) / gridDim.x;
    const uint32_t nch = (uint32_t)(c1 - c0), T = nch * GT_L;
    if (warp == GT_PRODUCERS + 4) {
        if (lane == 0) {
            mbar_init(bars + 0, 1);
            for (int i = 0; i < GT_RING; i++) { mbar_init(full + i, 4); mbar_init(empty + i, 1); }
            for (int i = 0; i < 2; i++) { mbar_init(accfull + i, 1); mbar_init(accempty + i, 4); }
            for (int i = 0; i < GT_STAGES; i++) { mbar_init(sfull + i, 1); mbar_init(sempty + i, 4); }
            mbar_expect_tx(bars + 0, GT_BMAT_TOTAL + KTAB_BYTES);
            for (int e = 0; e < GT_L; e++)
                bulk_copy_g2s(sm + GT_BMAT_OFF + e * TC_BMAT_BYTES, reinterpret_cast<const uint8_t *>(p.bmat2) + e * TC_BMAT_BYTES, TC_BMAT_BYTES, bars + 0);
            bulk_copy_g2s(sm + KTAB_OFF, p.ktab2, KTAB_BYTES, bars + 0);
        }
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tslot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    gt_fence_before();
    __syncthreads();
    gt_fence_after();
    const uint32_t tbase = *tslot;
    const uint32_t tb = __shfl_sync(0xFFFFFFFFu, tbase, 0);      // the same value, known to be warp-uniform
    if (warp < 4) {                                     // scale factors: every byte 2^0 (UE8M0 127)
        const uint32_t one = 0x7F7F7F7Fu, a = tbase + ((32u * warp) << 16) + GT_COL_SF;
#pragma unroll
        for (int c = 0; c < 32; c += 8)
            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(a + c), "r"(one) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    gt_fence_before();
    __syncthreads();
    gt_fence_after();

    if (warp < GT_PRODUCERS) {
        // ---- producers: slices tt = (warp >> 2) + NSUB i, rows 32 (warp & 3) .. + 31 -----------------------------------
        const uint32_t q = warp & 3, sub = warp >> 2;
        const uint32_t lanebase = tbase + ((32u * q) << 16);
        constexpr uint32_t NSUB = GT_PRODUCERS / 4;                    // slice tt belongs to the warps with sub == tt % NSUB
        const uint32_t n = T > sub ? (T - sub + NSUB - 1) / NSUB : 0;  // slices of this warp
        const uint32_t mine = smem_u32(sm + GT_STAGE_OFF) + 16 * (32 * q + lane);
        uint32_t slot = sub, ph = 1;                                   // ring position of this warp's next slice; parity to wait for
        uint32_t stage = sub, sph = 0;                                 // the same for the staging ring in shared memory
        for (uint32_t i = 0; i < n; i++) {
            mbar_wait(sfull + stage, sph);                             // the slice has landed (bulk copy)
            uint4 x;
            asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(x.x), "=r"(x.y), "=r"(x.z), "=r"(x.w) : "r"(mine + 2048 * stage) : "memory");
            uint32_t v[16];
            const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
            for (int c = 0; c < 4; c++) {
                v[4 * c + 0] = w[c] & 0x11111111u;                      // bits 0, 4, ..: e2m1 0.5
                v[4 * c + 1] = w[c] & 0x22222222u;                      // bits 1, 5, ..: 1.0
                v[4 * c + 2] = w[c] & 0x44444444u;                      // bits 2, 6, ..: 2.0
                v[4 * c + 3] = (w[c] >> 1) & 0x44444444u;               // bits 3, 7, ..: 2.0
            }
            __syncwarp();
            if (lane == 0) gt_arrive(sempty + stage);                  // this warp's quarter of the stage is in registers
            mbar_wait(empty + slot, ph);
            gt_fence_after();
            asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                         ::"r"(lanebase + GT_COL_RING + 16 * slot), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                           "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            gt_fence_before();
            __syncwarp();
            if (lane == 0) gt_arrive(full + slot);
            slot += NSUB;
            if (slot >= GT_RING) { slot -= GT_RING; ph ^= 1; }
            stage += NSUB;
            if (stage >= GT_STAGES) { stage -= GT_STAGES; sph ^= 1; }
        }
    } else if (warp == GT_PRODUCERS + 5) {
        // ---- the load warp: one bulk copy (TMA 1-D) per slice of 2 KB, GT_STAGES of them in flight.  Every lane walks the
        // loop (addresses stay warp-uniform: UBLKCP takes uniform registers), one elected lane issues -----------------
        const uint32_t st0 = smem_u32(sm + GT_STAGE_OFF), sf0 = smem_u32(sfull), se0 = smem_u32(sempty);
        const uint64_t n_full = p.len / 16, n_cb = (p.len + 15) / 16, last = p.nchunks * GT_CHUNK_BLOCKS - 1;
        const uint64_t v_run = c0 * GT_CHUNK_BLOCKS;                   // virtual index of the run's first block
        // slices [t_lo, t_hi) of the run hold whole blocks of C only and arrive by bulk copy; the (at most three) others,
        // at either end of the message, are put together by hand
        uint32_t t_lo = 0, t_hi = 0;
        {
            const uint64_t lo = p.base > v_run ? (p.base - v_run + 127) / 128 : 0;
            const uint64_t end = p.base + n_full;                       // first virtual block that is not a whole block of C
            const uint64_t hi = end > v_run ? (end - v_run) / 128 : 0;
            t_lo = (uint32_t)(lo < T ? lo : T);
            t_hi = (uint32_t)(hi < T ? hi : T);
            if (t_hi < t_lo) t_hi = t_lo;
        }
        pdl_wait();
        uint32_t stage = 0, sph = 1, sa = st0, fa = sf0, ea = se0;
        const uint8_t *src = p.in + 16 * (v_run + 128ull * t_lo - p.base);      // used from slice t_lo on
        uint32_t tt = 0;
        while (tt < T) {
            if (tt >= t_lo && tt < t_hi) {
#pragma unroll 1
                for (; tt < t_hi; tt++) {                               // the steady state: nothing but additions
                    mbar_wait_addr(ea, sph);
                    if (gt_elect()) {
                        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], 2048;" ::"r"(fa) : "memory");
                        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 2048, [%2];"
                                     ::"r"(sa), "l"(src), "r"(fa) : "memory");
                    }
                    __syncwarp();
                    src += 2048; sa += 2048; fa += 8; ea += 8;
                    if (++stage == GT_STAGES) { stage = 0; sph ^= 1; sa = st0; fa = sf0; ea = se0; }
                }
                continue;
            }
            mbar_wait_addr(ea, sph);
            const uint64_t v0 = v_run + 128ull * tt;
#pragma unroll 1
            for (uint32_t k = 0; k < 4; k++) {
                const uint64_t v = v0 + 32 * k + lane;
                uint4 x = make_uint4(0, 0, 0, 0);
                if (v == last) {                                        // a10: BE64(8 a) || BE64(8 len)
                    const uint64_t abits = p.aad_len * 8, cbits = p.len * 8;
                    x = make_uint4(bswap32((uint32_t)(abits >> 32)), bswap32((uint32_t)abits), bswap32((uint32_t)(cbits >> 32)), bswap32((uint32_t)cbits));
                } else if (v >= p.base) {
                    const uint64_t g = v - p.base;
                    if (g < n_cb) {
                        const uint64_t rem = p.len - 16 * g;
                        x = rem >= 16 ? __ldg(reinterpret_cast<const uint4 *>(p.in + 16 * g)) : load_bytes(p.in + 16 * g, (uint32_t)rem);
                    }
                } else if (v >= p.pad) {
                    const uint64_t u = v - p.pad, rem = p.aad_len - 16 * u;
                    x = load_bytes(p.aad + 16 * u, rem < 16 ? (uint32_t)rem : 16u);
                }
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(sa + 16 * (32 * k + lane)), "r"(x.x), "r"(x.y), "r"(x.z), "r"(x.w) : "memory");
            }
            __syncwarp();
            if (gt_elect()) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(fa) : "memory");
            __syncwarp();
            tt++;
            sa += 2048; fa += 8; ea += 8;
            if (++stage == GT_STAGES) { stage = 0; sph ^= 1; sa = st0; fa = sf0; ea = se0; }
        }
    } else if (warp == GT_PRODUCERS + 4) {
        // ---- the issuing warp: every lane walks the loop (so that addresses and descriptors are warp-uniform and live
        // in uniform registers: UTCOMMA takes no others), one elected lane issues -------------------------------------
        mbar_wait(bars + 0, 0);
        // Everything the loop needs is kept up to date by additions: the uniform datapath that feeds UTCOMMA is slow,
        // and an issue loop of more than 128 cycles per slice would hold the tensor pipe back.
        const uint32_t sf = tb + GT_COL_SF, ring0 = tb + GT_COL_RING;
        const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty);
        const uint64_t dtop = gt_smem_desc(smem_u32(sm + GT_BMAT_OFF) + (GT_L - 1) * TC_BMAT_BYTES, 2048, 128);   // matrix of K^(GT_L-1), first half
        const uint32_t dhi = (uint32_t)(dtop >> 32), dlo_top = (uint32_t)dtop;
        uint32_t slot0 = 0, ph0 = 0;                                   // ring position and phase at the start of the chunk
        for (uint32_t c = 0; c < nch; c++) {
            const uint32_t b = c & 1, d = tb + 128 * b;
            mbar_wait(accempty + b, ((c >> 1) & 1) ^ 1);               // the read-back of this buffer's previous chunk is done
            if (gt_elect()) {
                uint32_t dlo = dlo_top, slot = slot0, ph = ph0;
                uint32_t a = ring0 + 16 * slot, fa = full0 + 8 * slot, ea = empty0 + 8 * slot;
#pragma unroll 1
                for (uint32_t s = 0; s < GT_L; s += 4) {               // four slices per trip: offsets fold into the instructions
#pragma unroll
                    for (uint32_t k = 0; k < 4; k++) {
                        mbar_wait_addr(fa + 8 * k, ph);
                        gt_fence_after();
                        gt_mma(d, a + 16 * k, ((uint64_t)dhi << 32) | (dlo - 512 * k), sf, s + k);
                        gt_mma(d, a + 16 * k + 8, ((uint64_t)dhi << 32) | (dlo - 512 * k + 256), sf, 1);
                        gt_commit_addr(ea + 8 * k);
                    }
                    dlo -= 4 * (TC_BMAT_BYTES >> 4);                   // on to the next lower powers of K
                    a += 64; fa += 32; ea += 32; slot += 4;
                    if (slot == GT_RING) { slot = 0; ph ^= 1; a = ring0; fa = full0; ea = empty0; }
                }
                gt_commit(accfull + b);
            }
            __syncwarp();
            slot0 += GT_L;                                              // every lane keeps the chunk-level position
            while (slot0 >= GT_RING) { slot0 -= GT_RING; ph0 ^= 1; }
        }
    } else {
        // ---- read-back warps: row 32 q + lane -----------------------------------------------------------------------
        const uint32_t q = warp & 3;
        const uint32_t lanebase = tbase + ((32u * q) << 16);
        mbar_wait(bars + 0, 0);                                         // the multiplier table has landed
        const MulK8 mul(sm, lane);
        uint4 Y = make_uint4(0, 0, 0, 0);
        for (uint32_t c = 0; c < nch; c++) {
            const uint32_t b = c & 1;
            mbar_wait(accfull + b, (c >> 1) & 1);
            gt_fence_after();
            uint32_t r[32];
            uint4 Z;
            gt_ld32(lanebase + 128 * b + 0, r);  Z.x = gt_parity32(r);
            gt_ld32(lanebase + 128 * b + 32, r); Z.y = gt_parity32(r);
            gt_ld32(lanebase + 128 * b + 64, r); Z.z = gt_parity32(r);
            gt_ld32(lanebase + 128 * b + 96, r); Z.w = gt_parity32(r);
            gt_fence_before();
            __syncwarp();
            if (lane == 0) gt_arrive(accempty + b);
            Y = xor4(mul(Y), Z);
        }
        uint4 part = make_uint4(0, 0, 0, 0);
        if (nch) part = gf_mul_mem(Y, __ldg(p.hx + (128 - (32 * q + lane))));     // row j ends 128 - j blocks before the run does
        part = gt_warp_xor4(part);
        if (lane == 0) red[q] = part;
    }
    gt_fence_before();
    __syncthreads();
    gt_fence_after();
    if (warp != GT_PRODUCERS + 4) return;
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase) : "memory");
    unsigned ticket = 0;
    if (lane == 0) {
        uint4 acc = xor4(xor4(red[0], red[1]), xor4(red[2], red[3]));
        const uint64_t behind = (p.nchunks - c1) * GT_CHUNK_BLOCKS;
        if (behind && nch) acc = gf_mul_mem(acc, gt_pow(p.hx, behind));
        pdl_wait();
        p.partials[blockIdx.x] = acc;
        asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(ticket) : "l"(p.counter) : "memory");
    }
    ticket = __shfl_sync(0xFFFFFFFFu, ticket, 0);
    if (ticket != p.ticket_last) return;
    uint4 tot = make_uint4(0, 0, 0, 0);
    for (uint32_t j = lane; j < gridDim.x; j += 32) tot = xor4(tot, __ldcg(p.partials + j));
    tot = gt_warp_xor4(tot);
    if (lane == 0) {
        if (p.chain_in != nullptr) tot = xor4(tot, gf_mul_mem(*p.chain_in, gt_pow(p.hx, p.nchunks * GT_CHUNK_BLOCKS)));
        *p.chain_out = tot;
        if (p.pow_out != nullptr) *p.pow_out = gt_pow(p.hx, p.exp_next);
    }
}

// ---- tables, once per key: bmat2[e] = bit matrix of H^(128 e), e < GT_L (layout as in gcm_tc.cu); ktab2 = the 8-bit
// multiplier table of H^(128 GT_L) (layout of gcm_common.cuh) ------------------------------------------------------
__global__ void __launch_bounds__(128, 1)
gcm_ghash_tc_setup_kernel(const uint4 *hx, uint4 *bmat2, uint4 *ktab2)
{
    __shared__ uint4 prod[128];
    const uint32_t e = blockIdx.x, t = threadIdx.x;
    // blocks 0 .. GT_L - 1: a matrix each; block GT_L: the table
    const uint4 P = gt_pow(hx, 128ull * e);
    if (e < GT_L) {
        uint32_t u[4] = {0, 0, 0, 0};
        u[t >> 5] = 1u << (t & 31);
        prod[t] = gf_mul_mem(make_uint4(u[0], u[1], u[2], u[3]), P);
        __syncthreads();
        for (uint32_t o = t; o < 512; o += 128) {
            const uint32_t i = o >> 7, n = o & 127;
            uint32_t out[4] = {0, 0, 0, 0};
#pragma unroll
            for (uint32_t j = 0; j < 4; j++) {
                const uint32_t val = j == 0 ? 4u : (j == 1 ? 2u : 1u);
                for (uint32_t mm = 0; mm < 8; mm++) {
                    const uint4 pr = prod[32 * i + 4 * mm + j];
                    const uint32_t w[4] = {pr.x, pr.y, pr.z, pr.w};
                    if ((w[n >> 5] >> (n & 31)) & 1u) {
                        const uint32_t q = 8 * j + mm;
                        out[q >> 3] |= val << (4 * (q & 7));
                    }
                }
            }
            bmat2[e * 512 + o] = make_uint4(out[0], out[1], out[2], out[3]);
        }
    } else {
        // V_i = P . x^i ("mem" format); entry (pos, v) = XOR over the set bits b of v of V[8 pos + 7 - b]
        gf128 u = gf_zero();
        u.w[t >> 5] = 1u << (31 - (t & 31));
        prod[t] = gf_to_mem(gf_mul(u, gf_from_mem(P)));
        __syncthreads();
        for (uint32_t k = t; k < 4096; k += 128) {
            const uint32_t pos = k >> 8, v = k & 0xFF;
            uint4 acc = make_uint4(0, 0, 0, 0);
            for (int b = 0; b < 8; b++)
                if ((v >> b) & 1) acc = xor4(acc, prod[8 * pos + 7 - b]);
            ktab2[v * 16 + (pos >> 3) * 8 + (pos & 7)] = acc;
        }
    }
}

void launch_ghash_tc_setup(const uint4 *hx, uint4 *bmat2, uint4 *ktab2, cudaStream_t s)
{
    gcm_ghash_tc_setup_kernel<<<GT_L + 1, 128, 0, s>>>(hx, bmat2, ktab2);
}

cudaError_t launch_ghash_tc(int blocks, const uint8_t *aad, uint64_t aad_len, const uint8_t *in, uint64_t len, const uint4 *bmat2,
                            const uint4 *ktab2, const uint4 *hx, uint4 *partials, unsigned *counter, unsigned ticket_last, uint4 *out,
                            cudaStream_t s)
{
    static std::atomic<bool> configured[GCM_MAX_DEVICES];
    const void *kern = (const void *)gcm_ghash_tc_kernel;
    cudaError_t e = ensure_smem_attr(kern, configured, GT_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    GhashTcParams p;
    memset(&p, 0, sizeof(p));
    const uint64_t n_aad = (aad_len + 15) / 16, blocks_real = n_aad + (len + 15) / 16 + 1;
    p.nchunks = ghash_tc_chunks(aad_len, len);
    p.pad = p.nchunks * GT_CHUNK_BLOCKS - blocks_real;
    p.base = p.pad + n_aad;
    p.in = in; p.aad = aad; p.len = len; p.aad_len = aad_len;
    p.bmat2 = bmat2; p.ktab2 = ktab2; p.hx = hx;
    p.partials = partials; p.counter = counter; p.ticket_last = ticket_last;
    p.chain_out = out;
    void *args[] = {(void *)&p};
    return launch_with_pdl(kern, dim3(blocks), dim3(GT_THREADS), GT_SMEM_BYTES, s, args);
}
