// gcm_setup.cu -- steps a1 + a2 of SURVEY.md 8(a): key schedule, H = E_K(0^128), the powers of H
// and the multiplier table of the fixed stride power (the table of
// powers of the hash key is generated on the GPU).  One CTA, runs once per key.
// Not hot.  Everything is computed from definitions; no typed-in tables.
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_setup.cuh"

// ---- GF(2^8), modulus x^8 + x^4 + x^3 + x + 1 (FIPS-197 4.2) -------------------------------------
__device__ __forceinline__ uint32_t gf8_xtime(uint32_t a) { return ((a << 1) ^ ((a & 0x80) ? 0x1B : 0)) & 0xFF; }

__device__ uint32_t gf8_mul(uint32_t a, uint32_t b)
{
    uint32_t p = 0;
    for (int i = 0; i < 8; i++) {
        if (b & 1) p ^= a;
        a = gf8_xtime(a);
        b >>= 1;
    }
    return p;
}

// S(a) = Aff(a^254): a^-1 = a^(2^8 - 2), 0 -> 0 (FIPS-197 5.1.1)
__device__ uint32_t sbox_of(uint32_t a)
{
    uint32_t r = 1, base = a;
    for (int e = 254; e; e >>= 1) {
        if (e & 1) r = gf8_mul(r, base);
        base = gf8_mul(base, base);
    }
    uint32_t inv = a ? r : 0;
    uint32_t rot = inv | (inv << 8);
    // b_i = a_i ^ a_(i+4) ^ a_(i+5) ^ a_(i+6) ^ a_(i+7) ^ c_i  ==  a ^ rotl(a,1..4) ^ 0x63
    return (inv ^ (rot >> 7) ^ (rot >> 6) ^ (rot >> 5) ^ (rot >> 4) ^ 0x63) & 0xFF;
}

__device__ __forceinline__ uint32_t rotl32(uint32_t x, int n) { return __funnelshift_l(x, x, n); }

// One block through the cipher with the single (non-replicated) T0 table in shared memory;
// state and round keys are little-endian column words.  Setup only.
__device__ uint4 aes_encrypt_setup(const uint32_t *te0, const uint32_t *rk, int nr, uint4 in)
{
    uint32_t s0 = in.x ^ rk[0], s1 = in.y ^ rk[1], s2 = in.z ^ rk[2], s3 = in.w ^ rk[3];
    for (int r = 1; r < nr; r++) {
        uint32_t t0 = te0[s0 & 0xFF] ^ rotl32(te0[(s1 >> 8) & 0xFF], 8) ^ rotl32(te0[(s2 >> 16) & 0xFF], 16) ^ rotl32(te0[s3 >> 24], 24) ^ rk[4 * r + 0];
        uint32_t t1 = te0[s1 & 0xFF] ^ rotl32(te0[(s2 >> 8) & 0xFF], 8) ^ rotl32(te0[(s3 >> 16) & 0xFF], 16) ^ rotl32(te0[s0 >> 24], 24) ^ rk[4 * r + 1];
        uint32_t t2 = te0[s2 & 0xFF] ^ rotl32(te0[(s3 >> 8) & 0xFF], 8) ^ rotl32(te0[(s0 >> 16) & 0xFF], 16) ^ rotl32(te0[s1 >> 24], 24) ^ rk[4 * r + 2];
        uint32_t t3 = te0[s3 & 0xFF] ^ rotl32(te0[(s0 >> 8) & 0xFF], 8) ^ rotl32(te0[(s1 >> 16) & 0xFF], 16) ^ rotl32(te0[s2 >> 24], 24) ^ rk[4 * r + 3];
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;
    }
    // final round: SubBytes + ShiftRows + AddRoundKey; S(x) is byte 1 of T0[x]
#define SB(x) ((te0[(x) & 0xFF] >> 8) & 0xFF)
    uint4 o;
    o.x = (SB(s0) | (SB(s1 >> 8) << 8) | (SB(s2 >> 16) << 16) | (SB(s3 >> 24) << 24)) ^ rk[4 * nr + 0];
    o.y = (SB(s1) | (SB(s2 >> 8) << 8) | (SB(s3 >> 16) << 16) | (SB(s0 >> 24) << 24)) ^ rk[4 * nr + 1];
    o.z = (SB(s2) | (SB(s3 >> 8) << 8) | (SB(s0 >> 16) << 16) | (SB(s1 >> 24) << 24)) ^ rk[4 * nr + 2];
    o.w = (SB(s3) | (SB(s0 >> 8) << 8) | (SB(s1 >> 16) << 16) | (SB(s2 >> 24) << 24)) ^ rk[4 * nr + 3];
#undef SB
    return o;
}

// FIPS-197 5.2 key expansion on big-endian words w[], then converted to little-endian column words.
__device__ void key_expand_setup(const uint32_t *sbox, const uint32_t *key_le, int nk, int nr, uint32_t *rk_le)
{
    uint32_t w[60];
    for (int i = 0; i < nk; i++) w[i] = bswap32(key_le[i]);
    uint32_t rcon = 1;
    for (int i = nk; i < 4 * (nr + 1); i++) {
        uint32_t t = w[i - 1];
        if (i % nk == 0) {
            t = (t << 8) | (t >> 24);
            t = (sbox[t >> 24] << 24) | (sbox[(t >> 16) & 0xFF] << 16) | (sbox[(t >> 8) & 0xFF] << 8) | sbox[t & 0xFF];
            t ^= rcon << 24;
            rcon = gf8_xtime(rcon);
        } else if (nk == 8 && i % 8 == 4) {
            t = (sbox[t >> 24] << 24) | (sbox[(t >> 16) & 0xFF] << 16) | (sbox[(t >> 8) & 0xFF] << 8) | sbox[t & 0xFF];
        }
        w[i] = w[i - nk] ^ t;
    }
    for (int i = 0; i < 4 * (nr + 1); i++) rk_le[i] = bswap32(w[i]);
    for (int i = 4 * (nr + 1); i < 60; i++) rk_le[i] = 0;
}

// out[i] = base^i for i = 0..count, by doubling: level `span` fills (span, 2*span] from
// out[i - span] . out[span].  One CTA; global memory made visible by __syncthreads().
__device__ void power_table(uint4 *out, uint4 base, int count)
{
    if (threadIdx.x == 0) {
        out[0] = gf_to_mem(gf_one());
        if (count >= 1) out[1] = base;
    }
    __syncthreads();
    for (int span = 1; span < count; span <<= 1) {
        gf128 top = gf_from_mem(out[span]);
        for (int i = span + 1 + threadIdx.x; i <= 2 * span && i <= count; i += blockDim.x)
            out[i] = gf_to_mem(gf_mul(gf_from_mem(out[i - span]), top));
        __syncthreads();
    }
}

__global__ void __launch_bounds__(512, 1)
gcm_setup_kernel(SetupParams p)
{
    __shared__ uint32_t s_sbox[256];
    __shared__ uint32_t s_te0[256];
    __shared__ uint32_t s_rk[60];
    __shared__ uint4 s_v[128];
    const int t = threadIdx.x;

    // a1: S-box and T0 from the definition
    if (t < 256) {
        uint32_t s = sbox_of(t);
        uint32_t s2 = gf8_xtime(s), s3 = s2 ^ s;
        s_sbox[t] = s;
        uint32_t te = s2 | (s << 8) | (s << 16) | (s3 << 24);
        s_te0[t] = te;
        p.te0[t] = te;
    }
    __syncthreads();
    const int nk = p.key_bits / 32, nr = nk + 6;
    if (t == 0) {
        key_expand_setup(s_sbox, p.key, nk, nr, s_rk);
        for (int i = 0; i < 60; i++) p.rk[i] = s_rk[i];
    }
    __syncthreads();
    // a2: H = E_K(0^128)
    if (t == 0) {
        uint4 h = aes_encrypt_setup(s_te0, s_rk, nr, make_uint4(0, 0, 0, 0));
        p.h[0] = h;
    }
    __syncthreads();
    gcm_build_power_tables(p.h[0], p.hpow, p.hx, p.ktab, s_v);
}

// Everything that depends on H only: hpow[i] = H^i (i <= 32), the radix-512 position-weight powers
// hx[k*512 + j] = H^(j * 512^k), K = H^32 and the Shoup table of K.
__device__ void gcm_build_power_tables(uint4 h, uint4 *hpow, uint4 *hx, uint4 *ktab, uint4 *s_v)
{
    const int t = threadIdx.x;
    power_table(hpow, h, GCM_STRIDE);
    uint4 base = h;
    for (int k = 0; k < HX_DIGITS; k++) {
        uint4 *tab = hx + (k << HX_RADIX_BITS);
        power_table(tab, base, (1 << HX_RADIX_BITS) - 1);
        base = gf_mul_mem(tab[(1 << HX_RADIX_BITS) - 1], base);     // base^(512): next digit's base
        __syncthreads();
    }
    // V_i = K . x^i, i = 0..127 ("mem" format): the images of the basis vectors
    if (t < 128) {
        gf128 e = gf_zero();
        e.w[t >> 5] = 1u << (31 - (t & 31));
        s_v[t] = gf_to_mem(gf_mul(e, gf_from_mem(hpow[GCM_STRIDE])));
    }
    __syncthreads();
    // entry (P, v) = XOR over the set bits b of v of V[8P + 7 - b]  (bit 7 of a byte is the lowest power)
    for (int e = t; e < 4096; e += blockDim.x) {
        int P = e >> 8, v = e & 0xFF;
        uint4 acc = make_uint4(0, 0, 0, 0);
        for (int b = 0; b < 8; b++)
            if ((v >> b) & 1) acc = xor4(acc, s_v[8 * P + 7 - b]);
        ktab[v * 16 + (P >> 3) * 8 + (P & 7)] = acc;
    }
}

// Overwrite a buffer with zeros: key material on destroy, and the plaintext on authentication
// failure ("physically suppressed via memset").  If `status` is non-NULL the wipe
// happens only when *status != 0 (the asynchronous validation gate).
__global__ void gcm_wipe_kernel(uint8_t *dst, uint64_t len, const int *status)
{
    if (status != nullptr && *status == 0) return;
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    // 16-byte stores over the aligned middle, bytes at the ragged ends
    uint64_t head = (16 - ((uintptr_t)dst & 15)) & 15;
    if (head > len) head = len;
    uint64_t mid = (len - head) / 16;
    for (uint64_t k = i; k < head; k += stride) dst[k] = 0;
    uint4 *d4 = reinterpret_cast<uint4 *>(dst + head);
    for (uint64_t k = i; k < mid; k += stride) d4[k] = make_uint4(0, 0, 0, 0);
    for (uint64_t k = head + mid * 16 + i; k < len; k += stride) dst[k] = 0;
}

// The key-independent round table alone (the batched kernel expands its keys itself).
__global__ void gcm_te0_kernel(uint32_t *te0)
{
    const uint32_t t = threadIdx.x;
    const uint32_t s = sbox_of(t), s2 = gf8_xtime(s), s3 = s2 ^ s;
    te0[t] = s2 | (s << 8) | (s << 16) | (s3 << 24);
}

void launch_setup(const SetupParams &p, cudaStream_t s) { gcm_setup_kernel<<<1, 512, 0, s>>>(p); }
void launch_te0(uint32_t *te0, cudaStream_t s) { gcm_te0_kernel<<<1, 256, 0, s>>>(te0); }
void launch_wipe(uint8_t *dst, uint64_t len, const int *status, cudaStream_t s)
{
    if (len == 0) return;
    uint64_t want = (len / 16 + 255) / 256 + 1;
    unsigned blocks = (unsigned)(want < 1184 ? want : 1184);   // 148 SMs x 8
    gcm_wipe_kernel<<<blocks, 256, 0, s>>>(dst, len, status);
}
