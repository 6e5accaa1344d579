// gf128.cuh -- GF(2^128) helpers of the CUDA path (setup kernels, per-thread / per-warp power
// corrections, finalisation, the batched kernel's tree).  NOT the hot multiply: the hot multiply by
// the fixed stride power K = H^32 is table driven (gcm_fused.cu, gcm_batch.cu).  Shares nothing with
// oracle/.
//
// Field and bit order: SP 800-38D section 6.3 -- a 16-byte block is the polynomial whose x^0
// coefficient is the most significant bit of byte 0; modulus x^128 + x^7 + x^2 + x + 1.
// ("multiplication in the Galois Field GF(2^128)".)
//
// Two representations are used:
//   * "mem"  : uint4 holding the 16 bytes as four little-endian words, exactly what LDG.128 of a
//              ciphertext block returns.  XOR works directly on it.
//   * "canon": gf128 {w[0..3]}, w[0] = bytes 0..3 read big-endian, so bit 31 of w[0] is x^0 and
//              bit 0 of w[3] is x^127; "multiply by x" is a 128-bit right shift.
#pragma once
#include <stdint.h>

struct gf128 { uint32_t w[4]; };

__device__ __forceinline__ uint32_t bswap32(uint32_t x) { return __byte_perm(x, 0, 0x0123); }

__device__ __forceinline__ gf128 gf_from_mem(uint4 m)
{
    gf128 r;
    r.w[0] = bswap32(m.x); r.w[1] = bswap32(m.y); r.w[2] = bswap32(m.z); r.w[3] = bswap32(m.w);
    return r;
}

__device__ __forceinline__ uint4 gf_to_mem(gf128 a)
{
    return make_uint4(bswap32(a.w[0]), bswap32(a.w[1]), bswap32(a.w[2]), bswap32(a.w[3]));
}

__device__ __forceinline__ gf128 gf_zero() { gf128 r; r.w[0] = r.w[1] = r.w[2] = r.w[3] = 0; return r; }
__device__ __forceinline__ gf128 gf_one()  { gf128 r = gf_zero(); r.w[0] = 0x80000000u; return r; }

__device__ __forceinline__ gf128 gf_xor(gf128 a, gf128 b)
{
    gf128 r;
    r.w[0] = a.w[0] ^ b.w[0]; r.w[1] = a.w[1] ^ b.w[1]; r.w[2] = a.w[2] ^ b.w[2]; r.w[3] = a.w[3] ^ b.w[3];
    return r;
}

// a . x : shift the 128-bit string right by one, fold the dropped x^127 coefficient back with
// R = 0xE1 || 0^120 (x^128 = 1 + x + x^2 + x^7).
__device__ __forceinline__ gf128 gf_mulx(gf128 a)
{
    uint32_t carry = 0u - (a.w[3] & 1u);
    gf128 r;
    r.w[3] = __funnelshift_r(a.w[3], a.w[2], 1);
    r.w[2] = __funnelshift_r(a.w[2], a.w[1], 1);
    r.w[1] = __funnelshift_r(a.w[1], a.w[0], 1);
    r.w[0] = (a.w[0] >> 1) ^ (carry & 0xE1000000u);
    return r;
}

// ---- generic product ------------------------------------------------------------------------------
// sm_100a has no carry-less multiply instruction; the integer multiplier (IMAD.WIDE on the FMA pipe,
// idle in this library's kernels) does the work instead.  A 32 x 32 -> 64 bit carry-less product is
// sixteen integer products of operands thinned to every fourth bit: each product then has at most 8
// overlapping partial products per 4-bit slot, so no carry leaves a slot and the slot's lowest bit
// is the GF(2) coefficient.  The four residue classes are XORed separately and merged by bit-select.
__device__ __forceinline__ uint64_t clmul32(uint32_t x, uint32_t y)
{
    const uint32_t x0 = x & 0x11111111u, x1 = x & 0x22222222u, x2 = x & 0x44444444u, x3 = x & 0x88888888u;
    const uint32_t y0 = y & 0x11111111u, y1 = y & 0x22222222u, y2 = y & 0x44444444u, y3 = y & 0x88888888u;
    const uint64_t u0 = ((uint64_t)x0 * y0) ^ ((uint64_t)x1 * y3) ^ ((uint64_t)x2 * y2) ^ ((uint64_t)x3 * y1);
    const uint64_t u1 = ((uint64_t)x0 * y1) ^ ((uint64_t)x1 * y0) ^ ((uint64_t)x2 * y3) ^ ((uint64_t)x3 * y2);
    const uint64_t u2 = ((uint64_t)x0 * y2) ^ ((uint64_t)x1 * y1) ^ ((uint64_t)x2 * y0) ^ ((uint64_t)x3 * y3);
    const uint64_t u3 = ((uint64_t)x0 * y3) ^ ((uint64_t)x1 * y2) ^ ((uint64_t)x2 * y1) ^ ((uint64_t)x3 * y0);
    const uint64_t m5 = 0x5555555555555555ull, m3 = 0x3333333333333333ull;
    const uint64_t t01 = (u0 & m5) | (u1 & ~m5);      // residues 0,2 from u0 / 1,3 from u1
    const uint64_t t23 = (u2 & m5) | (u3 & ~m5);      // residues 0,2 from u2 / 1,3 from u3
    return (t01 & m3) | (t23 & ~m3);                  // residues 0,1 from t01 / 2,3 from t23
}

// 64 x 64 -> 128 bit carry-less product, one Karatsuba level; r[0] least significant word.
__device__ __forceinline__ void clmul64(uint32_t xh, uint32_t xl, uint32_t yh, uint32_t yl, uint32_t (&r)[4])
{
    const uint64_t hh = clmul32(xh, yh), ll = clmul32(xl, yl);
    const uint64_t mm = clmul32(xh ^ xl, yh ^ yl) ^ hh ^ ll;
    r[0] = (uint32_t)ll;
    r[1] = (uint32_t)(ll >> 32) ^ (uint32_t)mm;
    r[2] = (uint32_t)hh ^ (uint32_t)(mm >> 32);
    r[3] = (uint32_t)(hh >> 32);
}

// a . b in GF(2^128).  "canon" words are the 128-bit big-endian integer whose bit (127 - i) is the
// coefficient of x^i, so the plain carry-less product P of the two integers holds the coefficient of
// x^k at bit (254 - k): after one left shift the upper 128 bits are the canon form of degrees 0..127
// and the lower 128 bits the canon form of (degrees 128..254) / x^128, which is folded back with
// x^128 = 1 + x + x^2 + x^7 (multiplying by x^s is a right shift by s; the up to 7 bits that fall off
// are folded once more and then fit).  ~350 ALU + 144 IMAD.WIDE instructions, short dependency chains.
__device__ __forceinline__ gf128 gf_reduce256(const uint32_t (&p)[8])     // p[0] least significant
{
    // P << 1
    const uint32_t lo0 = __funnelshift_l(p[6], p[7], 1), lo1 = __funnelshift_l(p[5], p[6], 1);
    const uint32_t lo2 = __funnelshift_l(p[4], p[5], 1), lo3 = __funnelshift_l(p[3], p[4], 1);
    const uint32_t h0 = __funnelshift_l(p[2], p[3], 1), h1 = __funnelshift_l(p[1], p[2], 1);
    const uint32_t h2 = __funnelshift_l(p[0], p[1], 1), h3 = p[0] << 1;
    // Hi . (1 + x + x^2 + x^7): 128-bit right shifts by 1, 2, 7 (h0 is the most significant word)
    uint32_t o = (h3 << 31) ^ (h3 << 30) ^ (h3 << 25);
    o ^= (o >> 1) ^ (o >> 2) ^ (o >> 7);
    gf128 r;
    r.w[0] = lo0 ^ h0 ^ (h0 >> 1) ^ (h0 >> 2) ^ (h0 >> 7) ^ o;
    r.w[1] = lo1 ^ h1 ^ __funnelshift_r(h1, h0, 1) ^ __funnelshift_r(h1, h0, 2) ^ __funnelshift_r(h1, h0, 7);
    r.w[2] = lo2 ^ h2 ^ __funnelshift_r(h2, h1, 1) ^ __funnelshift_r(h2, h1, 2) ^ __funnelshift_r(h2, h1, 7);
    r.w[3] = lo3 ^ h3 ^ __funnelshift_r(h3, h2, 1) ^ __funnelshift_r(h3, h2, 2) ^ __funnelshift_r(h3, h2, 7);
    return r;
}

static __device__ __noinline__ gf128 gf_mul(gf128 a, gf128 b)
{
    uint32_t hh[4], ll[4], mm[4];
    clmul64(a.w[0], a.w[1], b.w[0], b.w[1], hh);
    clmul64(a.w[2], a.w[3], b.w[2], b.w[3], ll);
    clmul64(a.w[0] ^ a.w[2], a.w[1] ^ a.w[3], b.w[0] ^ b.w[2], b.w[1] ^ b.w[3], mm);
    uint32_t p[8];                                     // p[0] least significant
    p[0] = ll[0]; p[1] = ll[1];
    p[2] = ll[2] ^ mm[0] ^ hh[0] ^ ll[0];
    p[3] = ll[3] ^ mm[1] ^ hh[1] ^ ll[1];
    p[4] = hh[0] ^ mm[2] ^ hh[2] ^ ll[2];
    p[5] = hh[1] ^ mm[3] ^ hh[3] ^ ll[3];
    p[6] = hh[2]; p[7] = hh[3];
    return gf_reduce256(p);
}

// a . a: squaring over GF(2) only spreads the bits (bit j of the integer moves to bit 2j), then the
// same reduction.  Used for the H^(2^k) ladder of PAPER.md L197.
__device__ __forceinline__ uint64_t spread32(uint32_t x)
{
    uint64_t t = x;
    t = (t | (t << 16)) & 0x0000FFFF0000FFFFull;
    t = (t | (t << 8)) & 0x00FF00FF00FF00FFull;
    t = (t | (t << 4)) & 0x0F0F0F0F0F0F0F0Full;
    t = (t | (t << 2)) & 0x3333333333333333ull;
    t = (t | (t << 1)) & 0x5555555555555555ull;
    return t;
}
static __device__ __noinline__ gf128 gf_sqr(gf128 a)
{
    uint32_t p[8];
#pragma unroll
    for (int i = 0; i < 4; i++) {                      // a.w[3] is the least significant word
        const uint64_t t = spread32(a.w[3 - i]);
        p[2 * i] = (uint32_t)t;
        p[2 * i + 1] = (uint32_t)(t >> 32);
    }
    return gf_reduce256(p);
}

__device__ __forceinline__ uint4 xor4(uint4 a, uint4 b)
{
    return make_uint4(a.x ^ b.x, a.y ^ b.y, a.z ^ b.z, a.w ^ b.w);
}

// product of two "mem" blocks
__device__ __forceinline__ uint4 gf_mul_mem(uint4 a, uint4 b)
{
    return gf_to_mem(gf_mul(gf_from_mem(a), gf_from_mem(b)));
}
