// gcm_multi.cu -- many large messages under ONE key in ONE launch (config C3: FITS-sized HDUs through
// the batched API).  Same per-block work as gcm_fused.cu; what changes is the
// work distribution: launching the single-message kernel once per 64 MiB image leaves ~30 us per image
// of table fill, position-weight setup, tail imbalance and finishing exposed (20 % of the image's
// time).  Here the shared-memory tables are filled once, the rows of ALL messages are dealt to the
// warps in contiguous chunks (a warp's chunks may straddle a message boundary), and each chunk's
// weighted GHASH partial is XOR-accumulated into its message's 16-byte accumulator with atomics
// (XOR is the field addition: order does not matter).  The last CTA to finish turns every accumulator
// into a tag (length block, E_K(J0)) or a verdict (constant-time compare).
//
// The sum per message is still sum X_i . H^(N-i+1) (Eq. 1 regrouped; L272-L286).
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_device.cuh"
#include "gcm_multi.cuh"

// H^d for d < 2^36 from the radix-512 digit table (see gcm_fused.cu)
__device__ __forceinline__ uint4 multi_h_power(const uint4 *hx, uint64_t d, uint32_t lane)
{
    const uint32_t k = lane & 3;
    const uint32_t digit = (uint32_t)(d >> (HX_RADIX_BITS * k)) & ((1u << HX_RADIX_BITS) - 1);
    uint4 f = __ldg(hx + (k << HX_RADIX_BITS) + digit);
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
        uint4 g;
        g.x = __shfl_xor_sync(0xFFFFFFFFu, f.x, o); g.y = __shfl_xor_sync(0xFFFFFFFFu, f.y, o);
        g.z = __shfl_xor_sync(0xFFFFFFFFu, f.z, o); g.w = __shfl_xor_sync(0xFFFFFFFFu, f.w, o);
        f = gf_mul_mem(f, g);
    }
    return f;
}

template <int NR, int MODE>
__global__ void __launch_bounds__(MULTI_THREADS, 1)
gcm_multi_kernel(const __grid_constant__ MultiParams p)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    __shared__ bool s_last;
    const uint32_t t = threadIdx.x, lane = t & 31, lane4 = lane * 4;
    const uint32_t warp = __shfl_sync(0xFFFFFFFFu, t >> 5, 0);
    const uint32_t wg = blockIdx.x * (MULTI_THREADS / 32) + warp;

    {
        KtabRegs<MULTI_THREADS> kr;
        ktab_load<MULTI_THREADS>(kr, p.tab.ktab);
        fill_aes_tables<MULTI_THREADS>(sm, p.tab.te0);
        ktab_store<MULTI_THREADS>(kr, sm);
    }
    __syncthreads();

    uint32_t sel[8];
#pragma unroll
    for (int r = 0; r < 8; r++) sel[r] = ((lane + r) & 7) << 4;

    uint32_t c0 = 0, c1 = 0;
    if (wg < p.n_warps) { c0 = __ldg(p.warp_first + wg); c1 = __ldg(p.warp_first + wg + 1); }

#pragma unroll 1
    for (uint32_t c = c0; c < c1; c++) {
        const uint32_t mi = __ldg(&p.chunks[c].msg), r0 = __ldg(&p.chunks[c].r0), r1 = __ldg(&p.chunks[c].r1);
        const MultiMsg *m = p.msgs + mi;
        const uint8_t *in = m->in;
        uint8_t *out = m->out;
        const uint64_t base = m->base, vblocks = m->vblocks;
        const uint32_t fast_lo = m->fast_lo, fast_hi = m->fast_hi, ctr_delta = m->ctr_delta;
        const uint32_t S = m->rows;
        const bool tail_chunk = r1 == S;
        uint4 wpow = make_uint4(0, 0, 0, 0);
        if (!tail_chunk) wpow = multi_h_power(p.tab.hx, vblocks - 32ull * r1, lane);
        const CtrConst cc = ctr_const(p.rk, m->iv[0], m->iv[1], m->iv[2], sm, lane4);
        CtrCache cu = {0, 0, 0, 0};

        uint4 Y = make_uint4(0, 0, 0, 0);
        uint4 pre = make_uint4(0, 0, 0, 0);
        bool have_pre = false;
#pragma unroll 1
        for (uint32_t row = r0; row < r1; row++) {
            const uint64_t v = 32ull * row + lane;
            const bool fast = row >= fast_lo && row < fast_hi;
            uint4 x = make_uint4(0, 0, 0, 0);
            uint32_t cbytes = 0;
            uint64_t g = 0;
            bool valid = true;
            if (fast) {
                g = v - base;
                x = have_pre ? pre : ld16_stream(in + 16 * g);
                cbytes = 16;
                have_pre = row + 1 < r1 && row + 1 < fast_hi;
                if (have_pre) pre = ld16_stream(in + 16 * g + 512);
            } else {
                have_pre = false;
                valid = v < vblocks;
                const uint32_t pad = m->pad, n_aad = m->n_aad_blocks;
                if (valid && v >= pad) {
                    const uint64_t u = v - pad;
                    if (u < n_aad) {
                        const uint64_t rem = m->aad_len - 16 * u;
                        x = load_bytes(m->aad + 16 * u, rem < 16 ? (uint32_t)rem : 16u);
                    } else {
                        g = u - n_aad;
                        const uint64_t rem = m->len - 16 * g;
                        cbytes = rem < 16 ? (uint32_t)rem : 16u;
                        x = (cbytes == 16 && m->aligned) ? ld16_stream(in + 16 * g) : load_bytes(in + 16 * g, cbytes);
                    }
                }
            }
            const uint4 ym = ghash_mul_k(sm, sel, Y);                                   // a7
            const uint32_t ctr = (uint32_t)v + ctr_delta;                              // a4
            if (row == r0 || (ctr & 0xE0u) == 0) cu = ctr_cache(p.rk, sm, lane4, cc, ctr);
            const uint4 ks = aes_ctr_block<NR>(p.rk, sm, lane4, cc, cu, ctr);           // a5
            const uint4 y = xor4(x, ks);                                               // a6
            if (cbytes == 16 && (fast || m->aligned)) st16_stream(out + 16 * g, y);
            else if (cbytes) store_bytes(out + 16 * g, y, cbytes);
            uint4 X = x;
            if (MODE == MODE_ENCRYPT && cbytes) X = keep_bytes(y, cbytes);
            if (fast || valid) Y = xor4(ym, X);
        }

        // a8: lane correction, XOR over the warp, position weight of the chunk, into the message's accumulator
        const uint32_t rem = tail_chunk ? (uint32_t)(vblocks - 32ull * (S - 1)) : 32u;   // 1..32
        const uint32_t e = ((rem - lane - 1) & 31) + 1;
        uint4 part = gf_mul_mem(Y, __ldg(p.tab.hpow + e));
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) {
            part.x ^= __shfl_xor_sync(0xFFFFFFFFu, part.x, o); part.y ^= __shfl_xor_sync(0xFFFFFFFFu, part.y, o);
            part.z ^= __shfl_xor_sync(0xFFFFFFFFu, part.z, o); part.w ^= __shfl_xor_sync(0xFFFFFFFFu, part.w, o);
        }
        if (!tail_chunk) part = gf_mul_mem(part, wpow);
        if (lane == 0) {
            atomicXor(p.acc + 2 * mi, (unsigned long long)part.x | ((unsigned long long)part.y << 32));
            atomicXor(p.acc + 2 * mi + 1, (unsigned long long)part.z | ((unsigned long long)part.w << 32));
        }
    }

    // a9: last-CTA-done; a10 + a11 per message by the threads of that CTA
    __syncthreads();
    if (t == 0) {
        __threadfence();
        const unsigned ticket = atomicAdd(p.counter, 1u);
        s_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const uint4 h = __ldg(p.tab.h);
    for (uint32_t mi = t; mi < p.n_msgs; mi += MULTI_THREADS) {
        const MultiMsg *m = p.msgs + mi;
        const unsigned long long a0 = __ldcg(p.acc + 2 * mi), a1 = __ldcg(p.acc + 2 * mi + 1);
        const uint4 acc = make_uint4((uint32_t)a0, (uint32_t)(a0 >> 32), (uint32_t)a1, (uint32_t)(a1 >> 32));
        const uint64_t abits = m->aad_len * 8, cbits = m->len * 8;
        const uint4 L = make_uint4(bswap32((uint32_t)(abits >> 32)), bswap32((uint32_t)abits),
                                   bswap32((uint32_t)(cbits >> 32)), bswap32((uint32_t)cbits));
        const uint4 Sg = gf_mul_mem(xor4(acc, L), h);
        const uint4 ek = aes_encrypt_block<NR>(p.rk, sm, lane4, make_uint4(m->iv[0], m->iv[1], m->iv[2], 0x01000000u));
        const uint4 tag = xor4(Sg, ek);
        MultiResult *res = p.results + m->result;
        if (MODE == MODE_ENCRYPT) {
            res->tag[0] = tag.x; res->tag[1] = tag.y; res->tag[2] = tag.z; res->tag[3] = tag.w;
            res->status = 0;
        } else {
            const uint32_t diff = (tag.x ^ m->tag_expect[0]) | (tag.y ^ m->tag_expect[1]) |
                                  (tag.z ^ m->tag_expect[2]) | (tag.w ^ m->tag_expect[3]);
            res->status = diff != 0 ? 1 : 0;
        }
    }
}

// grid (x, n_msgs): zero-fill the output of every message whose verdict is "authentication failure"
__global__ void gcm_multi_wipe_kernel(const MultiMsg *msgs, const MultiResult *results, uint32_t n_msgs)
{
    const uint32_t mi = blockIdx.y;
    if (mi >= n_msgs) return;
    const MultiMsg *m = msgs + mi;
    if (results[m->result].status == 0) return;
    uint8_t *dst = m->out;
    const uint64_t len = m->len;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint64_t head = (16 - ((uintptr_t)dst & 15)) & 15;
    if (head > len) head = len;
    const uint64_t mid = (len - head) / 16;
    for (uint64_t k = i; k < head; k += stride) dst[k] = 0;
    uint4 *d4 = reinterpret_cast<uint4 *>(dst + head);
    for (uint64_t k = i; k < mid; k += stride) d4[k] = make_uint4(0, 0, 0, 0);
    for (uint64_t k = head + mid * 16 + i; k < len; k += stride) dst[k] = 0;
}

template <int NR, int MODE>
static cudaError_t launch_multi_one(int blocks, const MultiParams &p, cudaStream_t s)
{
    auto kern = gcm_multi_kernel<NR, MODE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, FUSED_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    kern<<<blocks, MULTI_THREADS, FUSED_SMEM_BYTES, s>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_multi(int nr, int mode, int blocks, const MultiParams &p, cudaStream_t s)
{
    if (nr == 10) return mode == MODE_ENCRYPT ? launch_multi_one<10, MODE_ENCRYPT>(blocks, p, s)
                                              : launch_multi_one<10, MODE_DECRYPT>(blocks, p, s);
    return mode == MODE_ENCRYPT ? launch_multi_one<14, MODE_ENCRYPT>(blocks, p, s)
                                : launch_multi_one<14, MODE_DECRYPT>(blocks, p, s);
}

void launch_multi_wipe(const MultiMsg *msgs, const MultiResult *results, uint32_t n_msgs, cudaStream_t s)
{
    if (n_msgs == 0) return;
    for (uint32_t off = 0; off < n_msgs; off += 65535) {
        const uint32_t cnt = n_msgs - off < 65535 ? n_msgs - off : 65535;
        gcm_multi_wipe_kernel<<<dim3(64, cnt), 256, 0, s>>>(msgs + off, results, cnt);
    }
}
