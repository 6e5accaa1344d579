// gf128.cuh -- GF(2^128) helpers of the CUDA path (setup kernels, per-thread power correction,
// finalisation).  NOT the hot multiply: the hot multiply by the fixed stride power is table driven
// (ghash_tab.cuh).  Shares nothing with oracle/.
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

// Generic product, bit-serial over the bits of a (x^0 first), v = b . x^i kept by gf_mulx.
// ~1500 ALU instructions; used O(1) times per thread per launch, never per block.
static __device__ __noinline__ gf128 gf_mul(gf128 a, gf128 b)
{
    gf128 z = gf_zero();
    gf128 v = b;
#pragma unroll 1
    for (int wi = 0; wi < 4; wi++) {
        uint32_t aw = a.w[wi];
#pragma unroll 4
        for (int i = 0; i < 32; i++) {
            uint32_t m = 0u - ((aw >> 31) & 1u);
            aw <<= 1;
            z.w[0] ^= v.w[0] & m; z.w[1] ^= v.w[1] & m; z.w[2] ^= v.w[2] & m; z.w[3] ^= v.w[3] & m;
            v = gf_mulx(v);
        }
    }
    return z;
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
