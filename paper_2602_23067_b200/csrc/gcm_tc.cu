// gcm_tc.cu -- the fused kernel with GHASH on the tensor cores (tcgen05 / TMEM, sm_100a).
//
// Same path as gcm_fused.cu (Eq. 1), same rows, same counters,
// same epilogue; only the leaf fold a7 differs.  gcm_fused.cu multiplies every block by K = H^32 through a 64 KB
// shared-memory table: 16 LDS.128 per block on the shared-memory data pipe, the unit that binds that kernel.  Here
// the multiply is what it is over GF(2): a 128 x 128 bit matrix applied to a 128-bit vector, with XOR as the sum.
//
//   * A lane's L consecutive blocks X_0 .. X_(L-1) (32 blocks apart, as before) and its running value Y form one
//     chunk:  Y' = Y.K^L  xor  X_0.K^(L-1)  xor ... xor  X_(L-1).K^0.  Over GF(2) this is ONE vector-matrix product
//     [Y | X_0 | ... | X_(L-1)] (128 (L+1) bits)  x  [M(K^L) ; M(K^(L-1)) ; ... ; M(K^0)]  ((L+1) 128 x 128 bits),
//     M(P) being the bit matrix of "multiply by P".  The 128 lanes of four warps are the 128 rows of a tcgen05.mma
//     tile; the matrices are the same for every lane, warp, CTA and message (they depend on the key only).
//   * The tensor core has no GF(2) type on sm_100a (mma.sync .b1 is emulated with IMMA, tcgen05 has no boolean kind),
//     but kind::mxf4 multiplies 4-bit floats exactly and accumulates in fp32: bits become e2m1 values, the
//     accumulator counts the ones, and the parity of the count is the XOR.  Counts stay below 2^11, far inside fp32.
//     A 128 x 128 x 64 mxf4 MMA takes 64 cycles (measured): 16,384 bit-products per SM-cycle = one GHASH block per
//     SM-cycle, on a pipe that does nothing else in this library.
//   * Bits are not moved one by one to nibbles.  x & 0x11111111 leaves eight message bits at nibble position 0,
//     which e2m1 reads as 0.5; & 0x22222222 as 1.0; & 0x44444444 as 2.0 (bit 3 is the sign: those bits are shifted
//     down by one first).  The matrix rows that meet those nibbles hold 2.0 / 1.0 / 0.5 / 0.5, so every product is
//     exactly 1.0.  Five ALU instructions per 32 message bits; the scale factors of the block-scaled kind are all 2^0.
//   * The expanded block goes from registers straight into TMEM (tcgen05.st) and is read from there as the A operand;
//     the matrices (8 KB per power, (L+1) powers) sit in shared memory as the B operand; the accumulators are 128
//     TMEM columns per group of four warps.  No shared-memory traffic per block apart from the matrix reads of the
//     tensor core itself.
//   * After the last slice of a chunk the four warps read their accumulator rows back (tcgen05.ld), take the parity
//     of the 128 counts (one FFMA that moves bit 0 to bit i, one LOP3 per count) and have Y' in registers: it is the
//     first slice of the next chunk.  At the end of the run Y is exactly what the table recurrence would have left,
//     and the epilogue of gcm_fused.cu (lane exponent, warp XOR, position weights, last-CTA-done) follows unchanged.
//
// Roles: 12 producer warps in 3 groups of 4 (warp & 3 selects the TMEM lane quarter a warp may touch) + 3 warps whose
// lane 0 issues the tcgen05.mma of one group each (the groups do not wait for one another).  Per group: one accumulator (128 columns), a ring of two A slices (16 columns
// each), mbarriers full[2] (4 producer arrivals), empty[2] and accfull (tcgen05.commit).  Every warp of the CTA runs
// the same number of rows (a run that is one row short starts with an empty row: zero blocks are free in GHASH), so
// the issuing lanes know the slice sequence without being told.
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_fused.cuh"
#include "gcm_tc.cuh"

#include "gcm_device.cuh"

#include <atomic>

#define TC_NW        12                              /* producer warps */
#define TC_NG        (TC_NW / 4)                     /* groups = issuing warps */
#define TC_THREADS   (32 * (TC_NW + TC_NG))
#define TC_BMAT_OFF  AES_TAB_BYTES
#define TC_RED_OFF   (TC_BMAT_OFF + TC_BMAT_TOTAL)
#define TC_WPOW_OFF  (TC_RED_OFF + 512)
#define TC_BAR_OFF   (TC_WPOW_OFF + 512)            /* tabbar, full[3][2], empty[3][2], accfull[3]: 16 x 8 B; TMEM base: 4 B */
#define TC_SMEM_BYTES (TC_BAR_OFF + 16 * 8 + 16)

// TMEM columns (512 allocated): accumulators [0, 384), scale factors [384, 416), A ring [416, 512)
#define TC_COL_SF    384
#define TC_COL_RING  416

// instruction descriptor, kind::mxf4 block-scaled: A, B = E2M1 (1), K-major, N = 128, UE8M0 scales, M = 128, K = 64
#define TC_IDESC ((1u << 7) | (1u << 10) | (16u << 17) | (1u << 23) | (8u << 24))

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool tc_elect()
{
    uint32_t pred;
    asm volatile("{ .reg .pred p; elect.sync _|p, 0xFFFFFFFF; selp.u32 %0, 1, 0, p; }" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tc_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// shared-memory matrix descriptor: no swizzle, K-major; 16-byte units
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | (1ull << 46);
}
// D[tmem] (+)= A[tmem] . B[smem]^T, 128 x 128 x 64, e2m1 operands, all scale factors 2^0
__device__ __forceinline__ void tc_mma(uint32_t d, uint32_t a, uint64_t b, uint32_t sf, uint32_t accumulate)
{
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %5, 0;\n"
                 "tcgen05.mma.cta_group::1.kind::mxf4.block_scale.block32 [%0], [%1], %2, %3, [%4], [%4], p;\n}"
                 ::"r"(d), "r"(a), "l"(b), "r"(TC_IDESC), "r"(sf), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tc_st16(uint32_t taddr, const uint32_t (&v)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                   "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                   "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// 32 counts (fp32, < 2^11) -> 32 parity bits.  c . 2^i + 2^23 has bit 0 of c at mantissa bit i: one FFMA (the FMA
// pipe is idle in this kernel) and one LOP3 per count, eleven counts per partial word.
__device__ __forceinline__ uint32_t tc_parity32(const uint32_t (&r)[32])
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

// GH policy of the row loop (gcm_device.cuh: gcm_rows_gh): the blocks go to the tensor core.
struct TensorGhash {
    uint32_t lanebase;      // TMEM address of this warp's lane quarter, column 0
    uint32_t ring;          // first column of this group's two A slices
    uint32_t acc;           // first column of this group's accumulator
    uint64_t *full, *empty, *accfull;
    uint32_t lane;
    uint32_t n;             // slices stored so far
    uint32_t in_chunk, ell, rows_left, chunk;
    bool pending;           // the last slice's tcgen05.st has not been waited for / announced yet
    bool owed;              // a finished chunk's result has not been read back yet
    uint4 Y;

    __device__ __forceinline__ TensorGhash(uint32_t tbase, uint32_t warp, uint32_t lane_, uint64_t *bars, uint32_t rows)
        : lane(lane_), n(0), in_chunk(0), chunk(0), pending(false), owed(false), Y(make_uint4(0, 0, 0, 0))
    {
        const uint32_t g = warp >> 2, q = warp & 3;
        lanebase = tbase + ((32u * q) << 16);
        ring = TC_COL_RING + 32 * g;
        acc = 128 * g;
        full = bars + 1 + 2 * g;
        empty = bars + 7 + 2 * g;
        accfull = bars + 13 + g;
        rows_left = rows;
        ell = rows < TC_L ? rows : TC_L;
    }
    // the previous slice is complete in TMEM: tell the issuing lane
    __device__ __forceinline__ void flush()
    {
        if (!pending) return;
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(full + ((n - 1) & 1));
        pending = false;
    }
    __device__ __forceinline__ void emit(uint4 x)
    {
        flush();
        const uint32_t slot = n & 1;
        mbar_wait(empty + slot, ((n >> 1) & 1) ^ 1);          // the MMAs that read this slot two slices ago are done
        tc_fence_after();
        uint32_t v[16];
        const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
        for (int i = 0; i < 4; i++) {
            v[4 * i + 0] = w[i] & 0x11111111u;                  // bits 0, 4, ..: e2m1 0.5
            v[4 * i + 1] = w[i] & 0x22222222u;                  // bits 1, 5, ..: 1.0
            v[4 * i + 2] = w[i] & 0x44444444u;                  // bits 2, 6, ..: 2.0
            v[4 * i + 3] = (w[i] >> 1) & 0x44444444u;           // bits 3, 7, ..: 2.0
        }
        tc_st16(lanebase + ring + 16 * slot, v);
        pending = true;
        n++;
    }
    // The chunk's accumulator row -> Y (and on into the next chunk as its first slice).  Called one row AFTER the
    // chunk's last slice was announced, i.e. behind the next row's AES: the MMAs have long finished by then.
    __device__ __forceinline__ void extract()
    {
        mbar_wait(accfull, chunk & 1);
        tc_fence_after();
        uint32_t r[32];
        tc_ld32(lanebase + acc + 0, r);  Y.x = tc_parity32(r);
        tc_ld32(lanebase + acc + 32, r); Y.y = tc_parity32(r);
        tc_ld32(lanebase + acc + 64, r); Y.z = tc_parity32(r);
        tc_ld32(lanebase + acc + 96, r); Y.w = tc_parity32(r);
        chunk++;
        owed = false;
    }
    __device__ __forceinline__ void pre() {}
    __device__ __forceinline__ void absorb(uint4 X, bool take)
    {
        if (owed) { extract(); emit(Y); }                       // the running value leads the new chunk
        emit(take ? X : make_uint4(0, 0, 0, 0));
        in_chunk++;
        rows_left--;
        if (in_chunk == ell) {                                  // chunk complete: announce its last slice now,
            flush();                                            // read the result back later
            owed = true;
            in_chunk = 0;
            ell = rows_left < TC_L ? rows_left : TC_L;
        }
    }
    __device__ __forceinline__ uint4 finish()
    {
        if (owed) extract();
        return Y;
    }
};

// GH policy for a single row off the tensor core: Y <- Y.K xor X with a generic product (lanes without a block keep Y).
struct ProductGhash {
    uint4 K, Y, ym;
    __device__ __forceinline__ ProductGhash(uint4 k, uint4 y0) : K(k), Y(y0), ym(y0) {}
    __device__ __forceinline__ void pre() { ym = gf_mul_mem(Y, K); }
    __device__ __forceinline__ void absorb(uint4 X, bool take) { if (take) Y = xor4(ym, X); }
};

__device__ __forceinline__ uint4 tc_warp_xor4(uint4 v)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        v.x ^= __shfl_xor_sync(0xFFFFFFFFu, v.x, o); v.y ^= __shfl_xor_sync(0xFFFFFFFFu, v.y, o);
        v.z ^= __shfl_xor_sync(0xFFFFFFFFu, v.z, o); v.w ^= __shfl_xor_sync(0xFFFFFFFFu, v.w, o);
    }
    return v;
}

// a8, first half (as cta_position_weights of gcm_fused.cu): D_w = H^(blocks behind the run of warp w) for the
// producer warps of this CTA, by one warp.
__device__ __forceinline__ void tc_position_weights(const GcmParams &p, uint32_t lane, uint4 *wpow)
{
    const uint64_t E = p.m.vblocks;
    const uint32_t S = p.m.rows, w = lane >> 1, half = lane & 1;
    const uint64_t wg = (uint64_t)blockIdx.x * TC_NW + w;
    const uint32_t r1 = (uint32_t)(((wg + 1) * S) / p.warps);
    const uint64_t d = (w < TC_NW && r1 < S) ? E - 32ull * r1 : 0;
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
    if (half == 0 && w < TC_NW) wpow[w] = f;
}

template <int NR, int MODE>
__global__ void __launch_bounds__(TC_THREADS, 1)
gcm_tc_kernel(const __grid_constant__ GcmParams p)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    __shared__ uint4 s_ekj0;
    const uint32_t t = threadIdx.x, lane = t & 31, lane4 = lane * 4;
    const uint32_t warp = __shfl_sync(0xFFFFFFFFu, t >> 5, 0);
    uint4 *red = reinterpret_cast<uint4 *>(sm + TC_RED_OFF);
    uint4 *wpow = reinterpret_cast<uint4 *>(sm + TC_WPOW_OFF);
    uint64_t *bars = reinterpret_cast<uint64_t *>(sm + TC_BAR_OFF);
    uint32_t *tslot = reinterpret_cast<uint32_t *>(sm + TC_BAR_OFF + 16 * 8);

    pdl_launch_dependents();
    // every warp of every CTA runs the same number of rows: ceil(S / W)
    const uint32_t S = p.m.rows;
    const uint32_t rmax = (S + p.warps - 1) / p.warps;
    uint32_t r0 = 0, r1 = 0;
    if (warp == TC_NW) {
        if (lane == 0) {
            mbar_init(bars + 0, 1);                                        // matrices landed
            for (int i = 1; i <= 6; i++) mbar_init(bars + i, 4);           // full[g][slot]: one arrival per producer warp
            for (int i = 7; i <= 15; i++) mbar_init(bars + i, 1);          // empty[g][slot], accfull[g]: tcgen05.commit
            mbar_expect_tx(bars + 0, TC_BMAT_TOTAL);
            for (int e = 0; e <= TC_L; e++)
                bulk_copy_g2s(sm + TC_BMAT_OFF + e * TC_BMAT_BYTES, reinterpret_cast<const uint8_t *>(p.tab.bmat) + e * TC_BMAT_BYTES,
                              TC_BMAT_BYTES, bars + 0);
        }
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tslot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    } else if (warp < TC_NW) {
        if (MODE != MODE_GHASH) fill_aes_tables<32 * TC_NW>(sm, p.te0, t);
        const uint64_t wg = (uint64_t)blockIdx.x * TC_NW + warp;
        r0 = __shfl_sync(0xFFFFFFFFu, (uint32_t)((wg * S) / p.warps), 0);
        r1 = __shfl_sync(0xFFFFFFFFu, (uint32_t)(((wg + 1) * S) / p.warps), 0);
        const uint32_t f0 = r0 > p.m.fast_lo ? r0 : p.m.fast_lo, f1 = r1 < p.m.fast_hi ? r1 : p.m.fast_hi;
#pragma unroll
        for (uint32_t k = 0; k < 2; k++)
            if (f0 + k < f1) prefetch_l2(p.m.in + 16 * (32ull * (f0 + k) + lane - p.m.base));
    }
    tc_fence_before();
    __syncthreads();                                    // AES tables stored, mbarriers initialised, TMEM allocated
    tc_fence_after();
    const uint32_t tbase = *tslot;

    // Scale factors (every byte 2^0, UE8M0 127) go into TMEM between two CTA barriers, as in gcm_tc2.cu: the issuing
    // warps wait only on the matrix copy and on the producers' full[] arrivals, and a warp whose run is short arrives
    // almost at once, so without the second barrier an MMA of group 1 or 2 could read column TC_COL_SF before the
    // quarter warps' tcgen05.st has landed there.
    if (warp < 4) {
        const uint32_t one = 0x7F7F7F7Fu, a = tbase + ((32u * warp) << 16) + TC_COL_SF;
#pragma unroll
        for (int c = 0; c < 32; c += 8)
            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(a + c), "r"(one) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();                                    // scale factors are in TMEM before any MMA can be issued
    tc_fence_after();

    if (warp >= TC_NW) {
        // ---- the issuing warp of group g: its slices in order.  Every lane walks the loop, so that addresses and
        // descriptors are warp-uniform and sit in uniform registers (UTCOMMA takes no others; from a single lane of a
        // divergent branch the compiler feeds it through R2UR + election loops); one elected lane issues ----------
        {
            const uint32_t tb = __shfl_sync(0xFFFFFFFFu, tbase, 0);
            const uint32_t g = warp - TC_NW;
            uint64_t *full = bars + 1 + 2 * g, *empty = bars + 7 + 2 * g;
            mbar_wait(bars + 0, 0);
            const uint32_t bm = smem_u32(sm + TC_BMAT_OFF), sf = tb + TC_COL_SF;
            uint32_t n = 0, left = rmax;
            for (uint32_t c = 0; left; c++) {
                const uint32_t ell = left < TC_L ? left : TC_L;
                left -= ell;
                const uint32_t nsl = ell + (c ? 1u : 0u);
                for (uint32_t j = 0; j < nsl; j++, n++) {
                    const uint32_t e = c ? ell - j : ell - 1 - j;         // power of K this slice is multiplied by
                    const uint32_t slot = n & 1;
                    const uint64_t b0 = tc_smem_desc(bm + e * TC_BMAT_BYTES, 2048, 128);
                    const uint64_t b1 = tc_smem_desc(bm + e * TC_BMAT_BYTES + 4096, 2048, 128);
                    mbar_wait(full + slot, (n >> 1) & 1);
                    tc_fence_after();
                    const uint32_t a = tb + TC_COL_RING + 32 * g + 16 * slot;
                    if (tc_elect()) {
                        tc_mma(tb + 128 * g, a, b0, sf, j != 0);
                        tc_mma(tb + 128 * g, a + 8, b1, sf, 1);
                        tc_commit(empty + slot);
                        if (j + 1 == nsl) tc_commit(bars + 13 + g);
                    }
                    __syncwarp();
                }
            }
        }
        __syncwarp();
        tc_fence_before();
        __syncthreads();                                // epilogue barrier of the producers: every tcgen05.ld is done
        tc_fence_after();
        if (warp == TC_NW) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase) : "memory");
        return;
    }

    // ---- producer warps ---------------------------------------------------------------------------------------
    if (warp == 0) tc_position_weights(p, lane, wpow);

    CtrConst cc = {0, 0, 0, 0};
    if (MODE != MODE_GHASH) {
        cc = ctr_const(p.rk, p.iv[0], p.iv[1], p.iv[2], sm, lane4);
        if (warp == TC_NW - 1) {                         // a3: E_K(J0)
            const CtrCache c1 = ctr_cache(p.rk, sm, lane4, cc, 1u);
            const uint4 ek = aes_ctr_block<NR>(p.rk, sm, lane4, cc, c1, 1u);
            if (lane == 0) s_ekj0 = ek;
        }
    }
    pdl_wait();
    if (MODE == MODE_DECRYPT && p.status_init && blockIdx.x == 0 && t == 0) *p.status = GCM_STATUS_PENDING;

    const ParamMsgView m{p.m};
    // The ragged last row of the message (rem < 32 blocks) stays off the tensor core: its lanes beyond the end must
    // NOT be multiplied by K there (lane_exponent counts on that), and one matrix serves all 128 lanes of a tile.
    // The warp that owns it folds that one row with a generic product instead.
    const uint32_t rem = (r0 < r1 && r1 == S) ? (uint32_t)(p.m.vblocks - 32ull * (S - 1)) : 32u;     // 1..32
    const uint32_t rt = rem < 32 ? r1 - 1 : r1;                  // rows [r0, rt) go through the tensor core
    TensorGhash gh(tbase, warp, lane, bars, rmax);
    for (uint32_t k = rt - r0; k < rmax; k++) gh.absorb(make_uint4(0, 0, 0, 0), false);   // a run that is short starts with empty rows
    gcm_rows_gh<NR, MODE, MODE == MODE_GHASH ? 2 : 1>(m, p.rk, sm, lane, cc, r0, rt, gh);  // a4-a7
    uint4 Y = gh.finish();
    if (rt < r1) {
        ProductGhash gl(__ldg(p.tab.hpow + GCM_STRIDE), Y);
        gcm_rows_gh<NR, MODE, 1>(m, p.rk, sm, lane, cc, rt, r1, gl);
        Y = gl.Y;
    }

    // a8, second half, a9, a11: as in gcm_fused.cu
    uint4 part = make_uint4(0, 0, 0, 0);
    if (r0 < r1) part = gf_mul_mem(Y, __ldg(p.tab.hpow + lane_exponent(rem, lane)));
    part = tc_warp_xor4(part);
    if (lane == 0) red[warp] = part;
    tc_fence_before();
    __syncthreads();
    if (warp != 0) return;
    uint4 acc = make_uint4(0, 0, 0, 0), wgt = make_uint4(0, 0, 0, 0);
    if (lane < TC_NW) { acc = red[lane]; wgt = wpow[lane]; }
    acc = tc_warp_xor4(gf_mul_mem(acc, wgt));
    unsigned ticket = 0;
    if (lane == 0) {
        p.partials[blockIdx.x] = acc;
        asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(ticket) : "l"(p.counter) : "memory");
    }
    ticket = __shfl_sync(0xFFFFFFFFu, ticket, 0);
    if (ticket != p.ticket_last) return;
    uint4 tot = make_uint4(0, 0, 0, 0);
    for (uint32_t j = lane; j < gridDim.x; j += 32) tot = xor4(tot, __ldcg(p.partials + j));
    tot = tc_warp_xor4(tot);
    if (lane == 0) {
        if (p.chain_in != nullptr) tot = xor4(tot, gf_mul_mem(*p.chain_in, *p.chain_pow));
        if (p.chain_out != nullptr) {
            *p.chain_out = tot;
        } else if (MODE == MODE_GHASH) {
            *p.tag_out = tot;
        } else {
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
}

// ---- the matrices (a2, once per key) ----------------------------------------------------------------------------
// bmat[e], e = 0 .. TC_L: the bit matrix of "multiply by K^e", K = H^32, as the B operand of the MMA: for message
// word i (0..3) and product bit n (0..127, bit n & 31 of word n >> 5, "mem" format) sixteen bytes = 32 nibbles;
// nibble 8 j + m belongs to message bit 4 m + j of word i and holds 2.0 / 1.0 / 0.5 / 0.5 (j = 0..3) where the
// matrix has a one.  [4][128][16 B] is the no-swizzle K-major core-matrix layout of two K = 64 MMAs (word pairs).
__global__ void __launch_bounds__(128, 1)
gcm_tc_setup_kernel(const uint4 *hx, uint4 *bmat)
{
    __shared__ uint4 prod[128];
    const uint32_t e = blockIdx.x, t = threadIdx.x;
    {
        uint32_t u[4] = {0, 0, 0, 0};
        u[t >> 5] = 1u << (t & 31);
        prod[t] = gf_mul_mem(make_uint4(u[0], u[1], u[2], u[3]), hx[GCM_STRIDE * e]);     // hx[j] = H^j, j < 512
    }
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
        bmat[e * 512 + o] = make_uint4(out[0], out[1], out[2], out[3]);
    }
}

void launch_tc_setup(const uint4 *hx, uint4 *bmat, cudaStream_t s)
{
    gcm_tc_setup_kernel<<<TC_L + 1, 128, 0, s>>>(hx, bmat);
}

template <int NR, int MODE>
static cudaError_t tc_launch_one(int blocks, const GcmParams &p, cudaStream_t s)
{
    static std::atomic<bool> configured[GCM_MAX_DEVICES];
    const void *kern = (const void *)gcm_tc_kernel<NR, MODE>;
    cudaError_t e = ensure_smem_attr(kern, configured, TC_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    void *args[] = {(void *)&p};
    return launch_with_pdl(kern, dim3(blocks), dim3(TC_THREADS), TC_SMEM_BYTES, s, args);
}

cudaError_t launch_tc(int nr, int mode, int blocks, const GcmParams &p, cudaStream_t s)
{
    if (mode == MODE_GHASH) return tc_launch_one<10, MODE_GHASH>(blocks, p, s);
    if (nr == 10) return mode == MODE_ENCRYPT ? tc_launch_one<10, MODE_ENCRYPT>(blocks, p, s) : tc_launch_one<10, MODE_DECRYPT>(blocks, p, s);
    return mode == MODE_ENCRYPT ? tc_launch_one<14, MODE_ENCRYPT>(blocks, p, s) : tc_launch_one<14, MODE_DECRYPT>(blocks, p, s);
}
