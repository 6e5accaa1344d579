// gcm_small.cu -- latency kernel for header-sized messages ("headers are typically small
// (< 80 kB), this provides low-latency access to metadata"; BASELINE config 4 measures single-message latency).
//
// A message of at most SMALL_MAX_BLOCKS GHASH blocks (AAD blocks + payload blocks + the length block: up to
// about 8 KiB) runs in ONE CTA with no cross-CTA step and no multiplier table: every block X_i is weighted
// directly by its own power of the hash key,
//     S = sum_i X_i . H^(N - i),   i = 0 .. N-1 over [AAD blocks | ciphertext blocks | length block],
// which is Eq. 1 written out; the powers H^1 .. H^511 are the first digit table of the
// context (hx[j] = H^j, built once per key by the setup kernel: "table of powers of the hash key", L197, L276).
// One generic GF(2^128) product per block on the integer multiplier, all blocks in parallel, then an XOR
// reduction: the depth is one AES block + one product + log2(threads) XORs whatever the length.
// The fused kernel's prologue (192 KB of tables, position weights, last-CTA-done hand-over) costs about 10 us
// however short the message is; this kernel fills the 128 KB AES tables only and finishes in about half that.
// Same arithmetic definitions, same counter rule (block g uses IV || BE32(g + 2)), shares nothing with oracle/.
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_fused.cuh"

#include "gcm_device.cuh"

#define SMALL_THREADS 256
#define SMALL_SMEM_BYTES (AES_TAB_BYTES + 512)

template <int NR, int MODE>
__global__ void __launch_bounds__(SMALL_THREADS, 1)
gcm_small_kernel(const __grid_constant__ GcmParams p)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    __shared__ uint4 s_ekj0;
    const uint32_t t = threadIdx.x, lane = t & 31, lane4 = lane * 4, warp = t >> 5;
    uint4 *red = reinterpret_cast<uint4 *>(sm + AES_TAB_BYTES);

    pdl_launch_dependents();
    pdl_wait();             // the payload loads below come first: nothing worth overlapping ahead of them
    // fail closed, as in gcm_fused.cu: a device-resident verdict word reads "refused" until thread 0 has compared the tags
    if (MODE == MODE_DECRYPT && p.status_init && t == 0 && p.chain_out == nullptr) *p.status = GCM_STATUS_PENDING;
    const uint32_t n_aad = p.m.n_aad_blocks;
    const uint32_t n_c = (uint32_t)((p.m.len + 15) / 16);
    const uint32_t N = n_aad + n_c + p.m.len_block;           // <= SMALL_MAX_BLOCKS (a link of a chunk chain may have no length block)
    const uint32_t ctr0 = (uint32_t)p.m.base + p.m.ctr_delta; // counter of payload block 0 of this launch: 2 + its index in the message

    // this thread's blocks (at most two) and their weights: global loads go out before the table fill
    uint4 x[2], w[2];
    uint32_t cbytes[2];
#pragma unroll
    for (int k = 0; k < 2; k++) {
        const uint32_t i = t + k * SMALL_THREADS;
        x[k] = make_uint4(0, 0, 0, 0);
        w[k] = make_uint4(0, 0, 0, 0);
        cbytes[k] = 0;
        if (i >= N) continue;
        w[k] = __ldg(p.tab.hx + (N - i));                     // H^(N - i), exponent 1 .. 511
        if (i < n_aad) {
            const uint64_t rem = p.m.aad_len - 16ull * i;
            x[k] = load_bytes(p.m.aad + 16ull * i, rem < 16 ? (uint32_t)rem : 16u);
        } else if (i < n_aad + n_c) {
            const uint32_t g = i - n_aad;
            const uint64_t rem = p.m.len - 16ull * g;
            cbytes[k] = rem < 16 ? (uint32_t)rem : 16u;
            x[k] = (cbytes[k] == 16 && p.m.aligned) ? ld16_stream(p.m.in + 16ull * g) : load_bytes(p.m.in + 16ull * g, cbytes[k]);
        } else {                                              // a10: BE64(8 a) || BE64(8 len)
            const uint64_t abits = p.m.final_aad_len * 8, cbits = p.m.final_len * 8;
            x[k] = make_uint4(bswap32((uint32_t)(abits >> 32)), bswap32((uint32_t)abits),
                              bswap32((uint32_t)(cbits >> 32)), bswap32((uint32_t)cbits));
        }
    }

    fill_aes_tables<SMALL_THREADS>(sm, p.te0, t);
    __syncthreads();

    // a3: E_K(J0), J0 = IV || 0^31 || 1, by the last warp; it reaches thread 0 through shared memory
    if (warp == SMALL_THREADS / 32 - 1) {
        const uint4 ek = aes_encrypt_block<NR>(p.rk, sm, lane4, make_uint4(p.iv[0], p.iv[1], p.iv[2], bswap32(1u)));
        if (lane == 0) s_ekj0 = ek;
    }

    uint4 acc = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int k = 0; k < 2; k++) {
        const uint32_t i = t + k * SMALL_THREADS;
        if (i >= N) continue;
        uint4 X = x[k];
        if (cbytes[k]) {                                      // a4-a6: payload block g, counter g + 2
            const uint32_t g = i - n_aad;
            const uint4 ks = aes_encrypt_block<NR>(p.rk, sm, lane4, make_uint4(p.iv[0], p.iv[1], p.iv[2], bswap32(g + ctr0)));
            const uint4 y = xor4(x[k], ks);
            if (cbytes[k] == 16 && p.m.aligned) st16_stream(p.m.out + 16ull * g, y);
            else store_bytes(p.m.out + 16ull * g, y, cbytes[k]);
            if (MODE == MODE_ENCRYPT) X = keep_bytes(y, cbytes[k]);
        }
        acc = xor4(acc, gf_mul_mem(X, w[k]));                 // a7: X_i . H^(N - i)
    }
    acc = cta_xor_reduce(acc, red);                           // a8 (no a9: one CTA)
    if (t == 0) {
        if (p.chain_in != nullptr) acc = xor4(acc, gf_mul_mem(*p.chain_in, *p.chain_pow));      // a link of a chunk chain (gcm_tc2.cu)
        if (p.chain_out != nullptr) { *p.chain_out = acc; return; }
        const uint4 tag = xor4(acc, s_ekj0);                  // a11
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

template <int NR, int MODE>
static cudaError_t launch_small_one(const GcmParams &p, cudaStream_t s)
{
    static std::atomic<bool> configured[GCM_MAX_DEVICES];
    const void *kern = (const void *)gcm_small_kernel<NR, MODE>;
    cudaError_t e = ensure_smem_attr(kern, configured, SMALL_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    void *args[] = {(void *)&p};
    return launch_with_pdl(kern, dim3(1), dim3(SMALL_THREADS), SMALL_SMEM_BYTES, s, args);
}

cudaError_t launch_small(int nr, int mode, const GcmParams &p, cudaStream_t s)
{
    if (nr == 10) return mode == MODE_ENCRYPT ? launch_small_one<10, MODE_ENCRYPT>(p, s) : launch_small_one<10, MODE_DECRYPT>(p, s);
    return mode == MODE_ENCRYPT ? launch_small_one<14, MODE_ENCRYPT>(p, s) : launch_small_one<14, MODE_DECRYPT>(p, s);
}
