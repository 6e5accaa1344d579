// gcm_device.cuh -- device helpers shared by the fused single-message kernel (gcm_fused.cu) and the
// batched many-message kernel (gcm_batch.cu): lane-replicated AES round tables in shared memory, the
// counter-block cipher with its per-thread / per-8-rows caches, byte-granular loads and stores for
// ragged ends, and the 8-bit Shoup multiply by the fixed stride power.  Shares nothing with oracle/.
#pragma once
#include "gcm_common.cuh"
#include "gf128.cuh"

__device__ __forceinline__ uint32_t lds32(const uint8_t *sm, uint32_t off)
{
    return *reinterpret_cast<const uint32_t *>(sm + off);
}
__device__ __forceinline__ uint4 lds128(const uint8_t *sm, uint32_t off)
{
    return *reinterpret_cast<const uint4 *>(sm + off);
}
__device__ __forceinline__ uint32_t rotl32(uint32_t x, int n) { return __funnelshift_l(x, x, n); }

// byte address of row (state byte `row` of w) in this lane's bank column: one PRMT
#define TIDX(w, row) __byte_perm((w), lane4, 0x5504u | ((row) << 4))

// Round-1 contribution of the three constant columns of a counter block (IV words ^ rk[0..2]):
// twelve of the sixteen round-1 table reads do not depend on the counter and are done once per thread.
struct CtrConst { uint32_t c0, c1, c2, c3; };

// RK: anything indexable that yields the round-key words rk[4r + c] (the kernel parameter block in
// the fused kernel: constant-bank operands; a register array in the batched kernel).
template <class RK>
__device__ __forceinline__ CtrConst ctr_const(const RK &rk, uint32_t iv0, uint32_t iv1, uint32_t iv2,
                                              const uint8_t *sm, uint32_t lane4)
{
    constexpr uint32_t T0 = AES_A0_OFF, T1 = AES_A0_OFF + AES_ODD_OFF, T2 = AES_A1_OFF, T3 = AES_A1_OFF + AES_ODD_OFF;
    const uint32_t s0 = iv0 ^ rk[0], s1 = iv1 ^ rk[1], s2 = iv2 ^ rk[2];   // IV words after AddRoundKey(0)
    CtrConst c;
    c.c0 = lds32(sm, TIDX(s0, 0) + T0) ^ lds32(sm, TIDX(s1, 1) + T1) ^ lds32(sm, TIDX(s2, 2) + T2) ^ rk[4];
    c.c1 = lds32(sm, TIDX(s1, 0) + T0) ^ lds32(sm, TIDX(s2, 1) + T1) ^ lds32(sm, TIDX(s0, 3) + T3) ^ rk[5];
    c.c2 = lds32(sm, TIDX(s2, 0) + T0) ^ lds32(sm, TIDX(s0, 2) + T2) ^ lds32(sm, TIDX(s1, 3) + T3) ^ rk[6];
    c.c3 = lds32(sm, TIDX(s0, 1) + T1) ^ lds32(sm, TIDX(s1, 2) + T2) ^ lds32(sm, TIDX(s2, 3) + T3) ^ rk[7];
    return c;
}

// Rounds 1-2 state that depends only on the upper 24 counter bits (see the header): the parts of the
// four round-2 output columns that do not come from round-1 column 0.
struct CtrCache { uint32_t u0, u1, u2, u3; };

template <class RK>
__device__ __forceinline__ CtrCache ctr_cache(const RK &rk, const uint8_t *sm, uint32_t lane4,
                                              const CtrConst &cc, uint32_t ctr)
{
    constexpr uint32_t T0 = AES_A0_OFF, T1 = AES_A0_OFF + AES_ODD_OFF, T2 = AES_A1_OFF, T3 = AES_A1_OFF + AES_ODD_OFF;
    const uint32_t c3 = bswap32(ctr) ^ rk[3];
    const uint32_t s1 = cc.c1 ^ lds32(sm, TIDX(c3, 2) + T2);
    const uint32_t s2 = cc.c2 ^ lds32(sm, TIDX(c3, 1) + T1);
    const uint32_t s3 = cc.c3 ^ lds32(sm, TIDX(c3, 0) + T0);
    CtrCache u;
    u.u0 = lds32(sm, TIDX(s1, 1) + T1) ^ lds32(sm, TIDX(s2, 2) + T2) ^ lds32(sm, TIDX(s3, 3) + T3) ^ rk[8];
    u.u1 = lds32(sm, TIDX(s1, 0) + T0) ^ lds32(sm, TIDX(s2, 1) + T1) ^ lds32(sm, TIDX(s3, 2) + T2) ^ rk[9];
    u.u2 = lds32(sm, TIDX(s2, 0) + T0) ^ lds32(sm, TIDX(s3, 1) + T1) ^ lds32(sm, TIDX(s1, 3) + T3) ^ rk[10];
    u.u3 = lds32(sm, TIDX(s3, 0) + T0) ^ lds32(sm, TIDX(s1, 2) + T2) ^ lds32(sm, TIDX(s2, 3) + T3) ^ rk[11];
    return u;
}

// E_K(IV || BE32(ctr)): a4 + a5.  Little-endian column words; the counter sits in column 3.  `u`
// must have been made by ctr_cache() from a counter with the same upper 24 bits.
template <int NR, class RK>
__device__ __forceinline__ uint4 aes_ctr_block(const RK &rk, const uint8_t *sm, uint32_t lane4,
                                               const CtrConst &cc, const CtrCache &u, uint32_t ctr)
{
    constexpr uint32_t T0 = AES_A0_OFF, T1 = AES_A0_OFF + AES_ODD_OFF, T2 = AES_A1_OFF, T3 = AES_A1_OFF + AES_ODD_OFF;
    // round 1: only column 0 depends on the low counter byte (state byte 15 = byte 3 of column 3)
    const uint32_t c3 = (ctr << 24) ^ rk[3];
    const uint32_t r0 = cc.c0 ^ lds32(sm, TIDX(c3, 3) + T3);
    // round 2: one read per column is indexed by round-1 column 0
    uint32_t s0 = u.u0 ^ lds32(sm, TIDX(r0, 0) + T0);
    uint32_t s1 = u.u1 ^ lds32(sm, TIDX(r0, 3) + T3);
    uint32_t s2 = u.u2 ^ lds32(sm, TIDX(r0, 2) + T2);
    uint32_t s3 = u.u3 ^ lds32(sm, TIDX(r0, 1) + T1);
#pragma unroll
    for (int r = 3; r < NR; r++) {
        uint32_t t0 = lds32(sm, TIDX(s0, 0) + T0) ^ lds32(sm, TIDX(s1, 1) + T1) ^ lds32(sm, TIDX(s2, 2) + T2) ^ lds32(sm, TIDX(s3, 3) + T3) ^ rk[4 * r + 0];
        uint32_t t1 = lds32(sm, TIDX(s1, 0) + T0) ^ lds32(sm, TIDX(s2, 1) + T1) ^ lds32(sm, TIDX(s3, 2) + T2) ^ lds32(sm, TIDX(s0, 3) + T3) ^ rk[4 * r + 1];
        uint32_t t2 = lds32(sm, TIDX(s2, 0) + T0) ^ lds32(sm, TIDX(s3, 1) + T1) ^ lds32(sm, TIDX(s0, 2) + T2) ^ lds32(sm, TIDX(s1, 3) + T3) ^ rk[4 * r + 2];
        uint32_t t3 = lds32(sm, TIDX(s3, 0) + T0) ^ lds32(sm, TIDX(s0, 1) + T1) ^ lds32(sm, TIDX(s1, 2) + T2) ^ lds32(sm, TIDX(s2, 3) + T3) ^ rk[4 * r + 3];
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;
    }
    // Final round (no MixColumns): S(x) sits in byte 0 of T2[x], bytes 1 and 2 of T0[x], byte 3 of T1[x].
    uint4 o;
#define FINAL(a, b, c, d, k)                                                                       \
    (__byte_perm(__byte_perm(lds32(sm, TIDX(a, 0) + T2), lds32(sm, TIDX(b, 1) + T0), 0x0050),      \
                 __byte_perm(lds32(sm, TIDX(c, 2) + T0), lds32(sm, TIDX(d, 3) + T1), 0x7200), 0x7610) ^ rk[4 * NR + (k)])
    o.x = FINAL(s0, s1, s2, s3, 0);
    o.y = FINAL(s1, s2, s3, s0, 1);
    o.z = FINAL(s2, s3, s0, s1, 2);
    o.w = FINAL(s3, s0, s1, s2, 3);
#undef FINAL
    return o;
}

// SubWord of FIPS-197 5.2 on a little-endian word, from the round tables.
__device__ __forceinline__ uint32_t aes_sub_word(const uint8_t *sm, uint32_t lane4, uint32_t x)
{
    constexpr uint32_t T0 = AES_A0_OFF, T1 = AES_A0_OFF + AES_ODD_OFF, T2 = AES_A1_OFF;
    return __byte_perm(__byte_perm(lds32(sm, TIDX(x, 0) + T2), lds32(sm, TIDX(x, 1) + T0), 0x0050),
                       __byte_perm(lds32(sm, TIDX(x, 2) + T0), lds32(sm, TIDX(x, 3) + T1), 0x7200), 0x7610);
}

// a1 inside a kernel: FIPS-197 5.2 key expansion on little-endian column words (RotWord is then a
// right rotation by 8 and Rcon lands in the low byte).  key: NK words as loaded from the key bytes.
template <int NR>
__device__ __forceinline__ void aes_key_expand(const uint8_t *sm, uint32_t lane4, const uint32_t *key,
                                               uint32_t (&rk)[4 * (NR + 1)])
{
    constexpr int NK = NR - 6;
#pragma unroll
    for (int i = 0; i < NK; i++) rk[i] = key[i];
    uint32_t rcon = 1;
#pragma unroll
    for (int i = NK; i < 4 * (NR + 1); i++) {
        uint32_t t = rk[i - 1];
        if (i % NK == 0) {
            t = aes_sub_word(sm, lane4, __funnelshift_r(t, t, 8)) ^ rcon;
            rcon = (rcon << 1) ^ ((rcon & 0x80u) ? 0x11Bu : 0u);       // x . rcon in GF(2^8)
        } else if (NK == 8 && i % 8 == 4) {
            t = aes_sub_word(sm, lane4, t);
        }
        rk[i] = rk[i - NK] ^ t;
    }
}

// E_K(in) for an arbitrary block (H = E_K(0), E_K(J0) in the batched kernel): no caches.
template <int NR, class RK>
__device__ __forceinline__ uint4 aes_encrypt_block(const RK &rk, const uint8_t *sm, uint32_t lane4, uint4 in)
{
    constexpr uint32_t T0 = AES_A0_OFF, T1 = AES_A0_OFF + AES_ODD_OFF, T2 = AES_A1_OFF, T3 = AES_A1_OFF + AES_ODD_OFF;
    uint32_t s0 = in.x ^ rk[0], s1 = in.y ^ rk[1], s2 = in.z ^ rk[2], s3 = in.w ^ rk[3];
#pragma unroll
    for (int r = 1; r < NR; r++) {
        uint32_t t0 = lds32(sm, TIDX(s0, 0) + T0) ^ lds32(sm, TIDX(s1, 1) + T1) ^ lds32(sm, TIDX(s2, 2) + T2) ^ lds32(sm, TIDX(s3, 3) + T3) ^ rk[4 * r + 0];
        uint32_t t1 = lds32(sm, TIDX(s1, 0) + T0) ^ lds32(sm, TIDX(s2, 1) + T1) ^ lds32(sm, TIDX(s3, 2) + T2) ^ lds32(sm, TIDX(s0, 3) + T3) ^ rk[4 * r + 1];
        uint32_t t2 = lds32(sm, TIDX(s2, 0) + T0) ^ lds32(sm, TIDX(s3, 1) + T1) ^ lds32(sm, TIDX(s0, 2) + T2) ^ lds32(sm, TIDX(s1, 3) + T3) ^ rk[4 * r + 2];
        uint32_t t3 = lds32(sm, TIDX(s3, 0) + T0) ^ lds32(sm, TIDX(s0, 1) + T1) ^ lds32(sm, TIDX(s1, 2) + T2) ^ lds32(sm, TIDX(s2, 3) + T3) ^ rk[4 * r + 3];
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;
    }
    uint4 o;
#define FINAL(a, b, c, d, k)                                                                       \
    (__byte_perm(__byte_perm(lds32(sm, TIDX(a, 0) + T2), lds32(sm, TIDX(b, 1) + T0), 0x0050),      \
                 __byte_perm(lds32(sm, TIDX(c, 2) + T0), lds32(sm, TIDX(d, 3) + T1), 0x7200), 0x7610) ^ rk[4 * NR + (k)])
    o.x = FINAL(s0, s1, s2, s3, 0);
    o.y = FINAL(s1, s2, s3, s0, 1);
    o.z = FINAL(s2, s3, s0, s1, 2);
    o.w = FINAL(s3, s0, s1, s2, 3);
#undef FINAL
    return o;
}

// y . K for the fixed stride power K: sixteen 16-byte table entries XORed (a7).  sel[r] =
// ((lane + r) & 7) << 4 is both the PRMT selector that moves byte (lane + r) & 7 of the 8-byte half
// into address byte 1 and the 16-byte column offset of that position inside the 128-byte half-row.
__device__ __forceinline__ uint4 ghash_mul_k(const uint8_t *sm, const uint32_t (&sel)[8], uint4 y)
{
    uint4 acc = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int r = 0; r < 8; r++) {
        uint32_t off = (__byte_perm(y.x, y.y, sel[r]) & 0xFF00u) | sel[r];
        acc = xor4(acc, lds128(sm, KTAB_OFF + off));
    }
#pragma unroll
    for (int r = 0; r < 8; r++) {
        uint32_t off = (__byte_perm(y.z, y.w, sel[r]) & 0xFF00u) | sel[r];
        acc = xor4(acc, lds128(sm, KTAB_OFF + 128 + off));
    }
    return acc;
}

__device__ __forceinline__ uint4 ld16_stream(const uint8_t *p)
{
    return __ldcs(reinterpret_cast<const uint4 *>(p));
}
__device__ __forceinline__ void st16_stream(uint8_t *p, uint4 v)
{
    __stcs(reinterpret_cast<uint4 *>(p), v);
}

// n (0..16) bytes -> block, zero-padded (a ragged tail, an unaligned buffer, an AAD block)
static __device__ __noinline__ uint4 load_bytes(const uint8_t *p, uint32_t n)
{
    uint32_t w[4] = {0, 0, 0, 0};
    uint32_t i = 0;
    if ((reinterpret_cast<uintptr_t>(p) & 3) == 0)          // whole words first when the pointer allows it
        for (; i + 4 <= n; i += 4) w[i >> 2] = *reinterpret_cast<const uint32_t *>(p + i);
    for (; i < n; i++) w[i >> 2] |= (uint32_t)p[i] << (8 * (i & 3));
    return make_uint4(w[0], w[1], w[2], w[3]);
}
static __device__ __noinline__ void store_bytes(uint8_t *p, uint4 v, uint32_t n)
{
    uint32_t w[4] = {v.x, v.y, v.z, v.w};
    for (uint32_t i = 0; i < n; i++) p[i] = (uint8_t)(w[i >> 2] >> (8 * (i & 3)));
}
// keep the first n bytes, zero the rest (GHASH sees the ciphertext zero-padded, never keystream)
__device__ __forceinline__ uint4 keep_bytes(uint4 v, uint32_t n)
{
    uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int k = 0; k < 4; k++) {
        int nb = (int)n - 4 * k;
        uint32_t m = nb >= 4 ? 0xFFFFFFFFu : (nb <= 0 ? 0u : ((1u << (8 * nb)) - 1u));
        w[k] &= m;
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}

// XOR of v over the CTA; result valid in thread 0.  red: 32 x uint4 of shared memory.
__device__ __forceinline__ uint4 cta_xor_reduce(uint4 v, uint4 *red)
{
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        v.x ^= __shfl_xor_sync(0xFFFFFFFFu, v.x, o); v.y ^= __shfl_xor_sync(0xFFFFFFFFu, v.y, o);
        v.z ^= __shfl_xor_sync(0xFFFFFFFFu, v.z, o); v.w ^= __shfl_xor_sync(0xFFFFFFFFu, v.w, o);
    }
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < nwarps ? red[lane] : make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) {
            v.x ^= __shfl_xor_sync(0xFFFFFFFFu, v.x, o); v.y ^= __shfl_xor_sync(0xFFFFFFFFu, v.y, o);
            v.z ^= __shfl_xor_sync(0xFFFFFFFFu, v.z, o); v.w ^= __shfl_xor_sync(0xFFFFFFFFu, v.w, o);
        }
    }
    __syncthreads();
    return v;
}

// AES table fill at kernel start, latency-critical for small and FITS-sized messages (Table A.7):
// the 1 KB round table T0 travels in the kernel parameter block (constant bank), so the expansion into the 128 KB
// lane-replicated layout needs no global load at all: one warp-uniform constant read and two 16-byte stores per
// four table words, 1024 store wavefronts per CTA in total.  Threads tid = 0 .. NT-1 share the work.
template <int NT, class TE0>
__device__ __forceinline__ void fill_aes_tables(uint8_t *sm, const TE0 &te0, uint32_t tid)
{
    uint4 *a0 = reinterpret_cast<uint4 *>(sm + AES_A0_OFF);
    uint4 *a1 = reinterpret_cast<uint4 *>(sm + AES_A1_OFF);
    // group g = four consecutive words of one 256-byte row (64 words: 32 x T_even | 32 x T_odd): 16 groups per row
#pragma unroll 4
    for (uint32_t g = tid; g < 4096; g += NT) {
        const uint32_t te = te0[g >> 4];
        const bool odd = (g >> 3) & 1;
        const uint32_t v0 = odd ? rotl32(te, 8) : te;                   // T0 | T1
        const uint32_t v1 = odd ? rotl32(te, 24) : rotl32(te, 16);      // T2 | T3
        a0[g] = make_uint4(v0, v0, v0, v0);
        a1[g] = make_uint4(v1, v1, v1, v1);
    }
}

// ---- sm_100a plumbing: bulk copy (TMA 1-D) completing on an mbarrier, programmatic dependent launch ----------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");      // visible to the async proxy
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completes on `bar` (SASS: UBLKCP)
__device__ __forceinline__ void bulk_copy_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// Programmatic dependent launch: the next kernel of the stream may start its prologue (table fill) while this
// grid drains; it must not touch stream-ordered data before pdl_wait().  Both are no-ops for a plain launch.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Pull a line towards L2 without returning data.  L2 is the coherence point of the device, so a line prefetched
// before griddepcontrol.wait stays correct even if the previous kernel of the stream still writes it.
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

__device__ __forceinline__ unsigned long long global_timer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// Shared-memory tables at kernel start.  The 64 KB GHASH multiplier table comes straight from the context slab by
// ONE bulk copy (TMA 1-D: cp.async.bulk, SASS UBLKCP) issued by thread 0 and completing on an mbarrier: no register
// staging, no store wavefronts; meanwhile the other threads expand the round table (above).  Reading the AES tables
// pre-expanded from L2 instead would move 128 KB per CTA x 148 CTAs = 19 MB through L2 per launch (2 us at the
// measured L2 rate) where the expansion costs 0.5 us of stores and no memory traffic.  With SPARE_WARP0 the first
// warp takes no part in the expansion (it has the position weights to form).  Call tables_wait() before the first
// table read.
template <int TPB, bool WITH_AES, bool SPARE_WARP0, class TE0>
__device__ __forceinline__ void tables_begin(uint8_t *sm, const GcmTables &tab, const TE0 &te0)
{
    uint64_t *bar = reinterpret_cast<uint64_t *>(sm + MBAR_OFF);
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_expect_tx(bar, KTAB_BYTES);
        bulk_copy_g2s(sm + KTAB_OFF, tab.ktab, KTAB_BYTES, bar);
    }
    if (WITH_AES) {
        if (SPARE_WARP0 && TPB > 32) {
            if (threadIdx.x >= 32) fill_aes_tables<TPB - 32>(sm, te0, threadIdx.x - 32);
        } else {
            fill_aes_tables<TPB>(sm, te0, threadIdx.x);
        }
    }
}
__device__ __forceinline__ void tables_wait(uint8_t *sm)
{
    __syncthreads();                                       // AES tables stored, mbarrier initialised
    mbar_wait(reinterpret_cast<uint64_t *>(sm + MBAR_OFF), 0);
}

// ---- GHASH multipliers for the row loop -----------------------------------------------------------------------
struct MulK8 {                 // 8-bit Shoup table of K in shared memory at KTAB_OFF (fused / multi kernels)
    const uint8_t *sm;
    uint32_t sel[8];
    __device__ __forceinline__ MulK8(const uint8_t *sm_, uint32_t lane) : sm(sm_)
    {
#pragma unroll
        for (int r = 0; r < 8; r++) sel[r] = ((lane + r) & 7) << 4;
    }
    __device__ __forceinline__ uint4 operator()(uint4 y) const { return ghash_mul_k(sm, sel, y); }
};

// ---- the row loop: SURVEY.md 8(a) a4-a7 for rows [r0, r1) of one message ------------------------------------
// MSG: accessor view of a RowMsg (hot fields in registers or constant bank, cold ones wherever they live).
// RK:  indexable round keys.  GH: the GHASH leaf fold (a7): gh.pre() before a row's AES, gh.absorb(X, take) with the
// row's GHASH input block after it (take = false: the lane has no block in this row).  TableGhash (below) multiplies
// by K through a shared-memory table (MUL: y -> y . K) and gcm_rows() returns its running value Y after the last
// block; TensorGhash (gcm_tc.cu) hands the blocks to the tensor core.
// The same code serves the single-message kernel (gcm_fused.cu), the many-large-messages kernel (gcm_multi.cu)
// and the warp-per-message kernel (gcm_batch.cu).
// DEPTH: rows of payload a lane keeps in flight ahead of the one it works on.  One row (512 B per warp, 8 KB per
// SM) covers the 1 TB/s the AES modes read; GHASH-only reads twice as fast and needs more bytes in flight to
// cover the HBM latency (Little's law: 2 TB/s x 0.8 us = 11 KB per SM).
template <int NR, int MODE, int DEPTH = 1, class MSG, class RK, class GH>
__device__ __forceinline__ void gcm_rows_gh(const MSG &m, const RK &rk, const uint8_t *sm, uint32_t lane,
                                            const CtrConst &cc, uint32_t r0, uint32_t r1, GH &gh)
{
    const uint32_t lane4 = lane * 4;
    CtrCache cu = {0, 0, 0, 0};
    uint4 pre = make_uint4(0, 0, 0, 0);
    bool have_pre = false;
    const uint32_t first_fast = r0 > m.fast_lo() ? r0 : m.fast_lo();      // first fast row of this run (if any)
    const uint32_t lim = r1 < m.fast_hi() ? r1 : m.fast_hi();             // fast rows of this run end here
    for (uint32_t row = r0; row < r1; row++) {
        const uint64_t v = 32ull * row + lane;          // virtual block index
        const bool fast = row >= m.fast_lo() && row < m.fast_hi();
        if (MODE == MODE_GHASH && DEPTH > 1 && fast && row == first_fast) {
            // GHASH only: all fast rows of the run in a DEPTH-deep software pipeline, unrolled DEPTH times so that
            // the slots keep their registers (no shifting); then on with the (slow) rows behind them
            const uint8_t *src = m.in() + 16 * (v - m.base());
            const uint32_t n = lim - row;
            uint4 buf[DEPTH];
#pragma unroll
            for (int k = 0; k < DEPTH; k++) buf[k] = (uint32_t)k < n ? ld16_stream(src + 512 * k) : make_uint4(0, 0, 0, 0);
            uint32_t i = 0;
            for (; i + DEPTH <= n; i += DEPTH) {
#pragma unroll
                for (int k = 0; k < DEPTH; k++) {
                    const uint4 xk = buf[k];
                    if (i + DEPTH + k < n) buf[k] = ld16_stream(src + 512ull * (i + DEPTH + k));
                    gh.pre();
                    gh.absorb(xk, true);
                }
            }
#pragma unroll
            for (int k = 0; k < DEPTH; k++)
                if (i + k < n) { gh.pre(); gh.absorb(buf[k], true); }
            row = lim - 1;
            continue;
        }
        uint4 x = make_uint4(0, 0, 0, 0);
        uint32_t cbytes = 0;                            // payload bytes in this block (0: pad / AAD / length block / beyond the end)
        uint64_t g = 0;                                 // payload block index
        bool valid = true;
        if (fast) {
            g = v - m.base();
            cbytes = 16;
            x = have_pre ? pre : ld16_stream(m.in() + 16 * g);
            have_pre = row + 1 < lim;
            if (have_pre) pre = ld16_stream(m.in() + 16 * g + 512);
        } else {
            have_pre = false;
            valid = v < m.vblocks();
            if (valid && v >= m.pad()) {
                const uint64_t u = v - m.pad();
                if (u < m.n_aad_blocks()) {
                    const uint64_t rem = m.aad_len() - 16 * u;
                    x = load_bytes(m.aad() + 16 * u, rem < 16 ? (uint32_t)rem : 16u);
                } else if (m.len_block() && v + 1 == m.vblocks()) {      // a10: BE64(8 a) || BE64(8 len)
                    const uint64_t abits = m.final_aad_len() * 8, cbits = m.final_len() * 8;
                    x = make_uint4(bswap32((uint32_t)(abits >> 32)), bswap32((uint32_t)abits),
                                   bswap32((uint32_t)(cbits >> 32)), bswap32((uint32_t)cbits));
                } else {
                    g = u - m.n_aad_blocks();
                    const uint64_t rem = m.len() - 16 * g;
                    cbytes = rem < 16 ? (uint32_t)rem : 16u;
                    x = (cbytes == 16 && m.aligned()) ? ld16_stream(m.in() + 16 * g) : load_bytes(m.in() + 16 * g, cbytes);
                }
            }
        }
        // a7: multiply the running value by K; independent of this row's AES, so they interleave
        gh.pre();
        uint4 X = x;
        if (MODE != MODE_GHASH) {
            // a4: counter from the virtual index alone; the upper 24 bits are warp-uniform and change
            // every 8th row, when rounds 1-2 are re-cached
            const uint32_t ctr = (uint32_t)v + m.ctr_delta();
            if (row == r0 || (ctr & 0xE0u) == 0) cu = ctr_cache(rk, sm, lane4, cc, ctr);
            const uint4 ks = aes_ctr_block<NR>(rk, sm, lane4, cc, cu, ctr);     // a5
            const uint4 y = xor4(x, ks);                                   // a6
            if (cbytes == 16 && (fast || m.aligned())) st16_stream(m.out() + 16 * g, y);
            else if (cbytes) store_bytes(m.out() + 16 * g, y, cbytes);
            if (MODE == MODE_ENCRYPT && cbytes) X = keep_bytes(y, cbytes);
        }
        gh.absorb(X, fast || valid);
    }
}

// GH for a table multiplier: Y <- Y.K xor X, the product formed ahead of the row's AES.
template <class MUL>
struct TableGhash {
    const MUL &mul;
    uint4 Y, ym;
    __device__ __forceinline__ explicit TableGhash(const MUL &mul_, uint4 y0 = make_uint4(0, 0, 0, 0)) : mul(mul_), Y(y0), ym(y0) {}
    __device__ __forceinline__ void pre() { ym = mul(Y); }
    __device__ __forceinline__ void absorb(uint4 X, bool take) { if (take) Y = xor4(ym, X); }
};

template <int NR, int MODE, int DEPTH = 1, class MSG, class RK, class MUL>
__device__ __forceinline__ uint4 gcm_rows(const MSG &m, const RK &rk, const uint8_t *sm, uint32_t lane,
                                          const CtrConst &cc, uint32_t r0, uint32_t r1, const MUL &mul)
{
    TableGhash<MUL> gh(mul);
    gcm_rows_gh<NR, MODE, DEPTH>(m, rk, sm, lane, cc, r0, r1, gh);
    return gh.Y;
}

// Exponent (1..32) of the power of H that aligns lane `lane`'s running value with the end of its run of rows:
// 32 - lane for a run that ends on a full row; in the ragged last row of the message (rem = 1..32 blocks) only
// lanes < rem folded a block there, and the lane order is rotated by rem.
__device__ __forceinline__ uint32_t lane_exponent(uint32_t rem, uint32_t lane) { return ((rem - lane - 1) & 31) + 1; }

// View of a RowMsg that lives in the kernel parameter block (constant bank): every field is a free operand.
struct ParamMsgView {
    const RowMsg &r;
    __device__ __forceinline__ const uint8_t *in() const { return r.in; }
    __device__ __forceinline__ uint8_t *out() const { return r.out; }
    __device__ __forceinline__ const uint8_t *aad() const { return r.aad; }
    __device__ __forceinline__ uint64_t len() const { return r.len; }
    __device__ __forceinline__ uint64_t aad_len() const { return r.aad_len; }
    __device__ __forceinline__ uint64_t base() const { return r.base; }
    __device__ __forceinline__ uint64_t vblocks() const { return r.vblocks; }
    __device__ __forceinline__ uint64_t final_len() const { return r.final_len; }
    __device__ __forceinline__ uint64_t final_aad_len() const { return r.final_aad_len; }
    __device__ __forceinline__ uint32_t pad() const { return r.pad; }
    __device__ __forceinline__ uint32_t n_aad_blocks() const { return r.n_aad_blocks; }
    __device__ __forceinline__ uint32_t fast_lo() const { return r.fast_lo; }
    __device__ __forceinline__ uint32_t fast_hi() const { return r.fast_hi; }
    __device__ __forceinline__ uint32_t aligned() const { return r.aligned; }
    __device__ __forceinline__ uint32_t ctr_delta() const { return r.ctr_delta; }
    __device__ __forceinline__ uint32_t len_block() const { return r.len_block; }
};

// View of a RowMsg in global memory: the fields the fast path touches are copied to registers once per chunk,
// the others are loaded where the slow path needs them.
struct GlobalMsgView {
    const RowMsg *g;
    const uint8_t *in_;
    uint8_t *out_;
    uint64_t base_;
    uint32_t fast_lo_, fast_hi_, ctr_delta_;
    __device__ __forceinline__ explicit GlobalMsgView(const RowMsg *p)
        : g(p), in_(p->in), out_(p->out), base_(p->base), fast_lo_(p->fast_lo), fast_hi_(p->fast_hi), ctr_delta_(p->ctr_delta) {}
    __device__ __forceinline__ const uint8_t *in() const { return in_; }
    __device__ __forceinline__ uint8_t *out() const { return out_; }
    __device__ __forceinline__ const uint8_t *aad() const { return g->aad; }
    __device__ __forceinline__ uint64_t len() const { return g->len; }
    __device__ __forceinline__ uint64_t aad_len() const { return g->aad_len; }
    __device__ __forceinline__ uint64_t base() const { return base_; }
    __device__ __forceinline__ uint64_t vblocks() const { return g->vblocks; }
    __device__ __forceinline__ uint64_t final_len() const { return g->final_len; }
    __device__ __forceinline__ uint64_t final_aad_len() const { return g->final_aad_len; }
    __device__ __forceinline__ uint32_t pad() const { return g->pad; }
    __device__ __forceinline__ uint32_t n_aad_blocks() const { return g->n_aad_blocks; }
    __device__ __forceinline__ uint32_t fast_lo() const { return fast_lo_; }
    __device__ __forceinline__ uint32_t fast_hi() const { return fast_hi_; }
    __device__ __forceinline__ uint32_t aligned() const { return g->aligned; }
    __device__ __forceinline__ uint32_t ctr_delta() const { return ctr_delta_; }
    __device__ __forceinline__ uint32_t len_block() const { return g->len_block; }
};

// View of a RowMsg held in registers (the warp-per-message kernel derives it from its descriptor).
struct RegMsgView {
    RowMsg r;
    __device__ __forceinline__ const uint8_t *in() const { return r.in; }
    __device__ __forceinline__ uint8_t *out() const { return r.out; }
    __device__ __forceinline__ const uint8_t *aad() const { return r.aad; }
    __device__ __forceinline__ uint64_t len() const { return r.len; }
    __device__ __forceinline__ uint64_t aad_len() const { return r.aad_len; }
    __device__ __forceinline__ uint64_t base() const { return r.base; }
    __device__ __forceinline__ uint64_t vblocks() const { return r.vblocks; }
    __device__ __forceinline__ uint64_t final_len() const { return r.final_len; }
    __device__ __forceinline__ uint64_t final_aad_len() const { return r.final_aad_len; }
    __device__ __forceinline__ uint32_t pad() const { return r.pad; }
    __device__ __forceinline__ uint32_t n_aad_blocks() const { return r.n_aad_blocks; }
    __device__ __forceinline__ uint32_t fast_lo() const { return r.fast_lo; }
    __device__ __forceinline__ uint32_t fast_hi() const { return r.fast_hi; }
    __device__ __forceinline__ uint32_t aligned() const { return r.aligned; }
    __device__ __forceinline__ uint32_t ctr_delta() const { return r.ctr_delta; }
    __device__ __forceinline__ uint32_t len_block() const { return r.len_block; }
};

