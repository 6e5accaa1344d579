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

// Table fill at kernel start, latency-critical for small messages (header-sized messages): all
// global loads of a thread are issued before its first shared-memory store, so the fill costs about one L2
// round trip plus the 1536 store wavefronts of the 192 KB, instead of one round trip per loop iteration.
template <int TPB>
__device__ __forceinline__ void fill_aes_tables(uint8_t *sm, const uint32_t *te0)
{
    uint32_t *a0 = reinterpret_cast<uint32_t *>(sm + AES_A0_OFF);
    uint32_t *a1 = reinterpret_cast<uint32_t *>(sm + AES_A1_OFF);
    constexpr int ROWS = (256 * 64 + TPB - 1) / TPB;       // table words per thread and array
    uint32_t te[ROWS];
#pragma unroll
    for (int k = 0; k < ROWS; k++) {
        const uint32_t j = threadIdx.x + k * TPB;
        te[k] = j < 16384 ? __ldg(te0 + (j >> 6)) : 0u;
    }
#pragma unroll
    for (int k = 0; k < ROWS; k++) {
        const uint32_t j = threadIdx.x + k * TPB;
        if (j < 16384) {
            const bool odd = (j >> 5) & 1;
            a0[j] = odd ? rotl32(te[k], 8) : te[k];                 // T0 | T1
            a1[j] = odd ? rotl32(te[k], 24) : rotl32(te[k], 16);    // T2 | T3
        }
    }
}

// The GHASH multiplier table: global loads into registers first (ktab_load), stores after the AES tables
// have been written (ktab_store), so the two fills share one memory round trip.
template <int TPB>
struct KtabRegs { uint4 v[(KTAB_BYTES / 16 + TPB - 1) / TPB]; };

template <int TPB>
__device__ __forceinline__ void ktab_load(KtabRegs<TPB> &r, const uint4 *ktab)
{
#pragma unroll
    for (int k = 0; k < (int)(sizeof(r.v) / sizeof(uint4)); k++) {
        const uint32_t j = threadIdx.x + k * TPB;
        r.v[k] = j < KTAB_BYTES / 16 ? __ldg(ktab + j) : make_uint4(0, 0, 0, 0);
    }
}
template <int TPB>
__device__ __forceinline__ void ktab_store(const KtabRegs<TPB> &r, uint8_t *sm)
{
    uint4 *kt = reinterpret_cast<uint4 *>(sm + KTAB_OFF);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(r.v) / sizeof(uint4)); k++) {
        const uint32_t j = threadIdx.x + k * TPB;
        if (j < KTAB_BYTES / 16) kt[j] = r.v[k];
    }
}
