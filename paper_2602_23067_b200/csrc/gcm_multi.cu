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
#include "gcm_fused.cuh"

// H^d for d < 2^36 from the radix-512 digit table (PAPER.md L197 precomputes H^(2^k): 36 factors; radix 512 needs
// 4): every lane of the warp takes part (lane & 3 picks the digit) and lanes with lane & 3 == 0 end up with the
// product.  d_max (a bound on d that is uniform over the warp) says how many digits can be non-zero.
__device__ __forceinline__ uint4 multi_h_power(const uint4 *hx, uint64_t d, uint32_t lane, uint64_t d_max)
{
    const uint32_t k = lane & 3;
    const uint32_t digit = (uint32_t)(d >> (HX_RADIX_BITS * k)) & ((1u << HX_RADIX_BITS) - 1);
    uint4 f = __ldg(hx + (k << HX_RADIX_BITS) + digit);
    const int levels = d_max < (1ull << HX_RADIX_BITS) ? 0 : (d_max < (1ull << (2 * HX_RADIX_BITS)) ? 1 : 2);
    for (int o = 1; o <= levels; o++) {
        const int mask = 1 << (o - 1);
        uint4 g;
        g.x = __shfl_xor_sync(0xFFFFFFFFu, f.x, mask); g.y = __shfl_xor_sync(0xFFFFFFFFu, f.y, mask);
        g.z = __shfl_xor_sync(0xFFFFFFFFu, f.z, mask); g.w = __shfl_xor_sync(0xFFFFFFFFu, f.w, mask);
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

    tables_begin<MULTI_THREADS, true, false>(sm, p.tab, p.te0);
    tables_wait(sm);
    const MulK8 mul(sm, lane);

    uint32_t c0 = 0, c1 = 0;
    if (wg < p.n_warps) { c0 = __ldg(p.warp_first + wg); c1 = __ldg(p.warp_first + wg + 1); }

#pragma unroll 1
    for (uint32_t c = c0; c < c1; c++) {
        const uint32_t mi = __ldg(&p.chunks[c].msg), r0 = __ldg(&p.chunks[c].r0), r1 = __ldg(&p.chunks[c].r1);
        const MultiMsg *mm = p.msgs + mi;
        const GlobalMsgView m(&mm->m);
        const uint64_t vblocks = mm->m.vblocks;
        const uint32_t S = mm->m.rows;
        const bool tail_chunk = r1 == S;
        uint4 wpow = make_uint4(0, 0, 0, 0);
        if (!tail_chunk) wpow = multi_h_power(p.tab.hx, vblocks - 32ull * r1, lane, vblocks);
        const CtrConst cc = ctr_const(p.rk, mm->iv[0], mm->iv[1], mm->iv[2], sm, lane4);

        const uint4 Y = gcm_rows<NR, MODE>(m, p.rk, sm, lane, cc, r0, r1, mul);         // a4-a7

        // a8: lane correction, XOR over the warp, position weight of the chunk, into the message's accumulator
        const uint32_t rem = tail_chunk ? (uint32_t)(vblocks - 32ull * (S - 1)) : 32u;   // 1..32
        uint4 part = gf_mul_mem(Y, __ldg(p.tab.hpow + lane_exponent(rem, lane)));
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

    // a9: last-CTA-done; a11 per message by the threads of that CTA (a10, the length block, was hashed by the rows)
    __syncthreads();
    if (t == 0) {
        __threadfence();
        const unsigned ticket = atomicAdd(p.counter, 1u);
        s_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (uint32_t mi = t; mi < p.n_msgs; mi += MULTI_THREADS) {
        const MultiMsg *mm = p.msgs + mi;
        const unsigned long long a0 = __ldcg(p.acc + 2 * mi), a1 = __ldcg(p.acc + 2 * mi + 1);
        const uint4 Sg = make_uint4((uint32_t)a0, (uint32_t)(a0 >> 32), (uint32_t)a1, (uint32_t)(a1 >> 32));
        const uint4 ek = aes_encrypt_block<NR>(p.rk, sm, lane4, make_uint4(mm->iv[0], mm->iv[1], mm->iv[2], 0x01000000u));
        const uint4 tag = xor4(Sg, ek);
        MultiResult *res = p.results + mm->result;
        if (MODE == MODE_ENCRYPT) {
            res->tag[0] = tag.x; res->tag[1] = tag.y; res->tag[2] = tag.z; res->tag[3] = tag.w;
            res->status = 0;
        } else {
            const uint32_t diff = (tag.x ^ mm->tag_expect[0]) | (tag.y ^ mm->tag_expect[1]) |
                                  (tag.z ^ mm->tag_expect[2]) | (tag.w ^ mm->tag_expect[3]);
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
    uint8_t *dst = m->m.out;
    const uint64_t len = m->m.len;
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
    static std::atomic<bool> configured[GCM_MAX_DEVICES];
    auto kern = gcm_multi_kernel<NR, MODE>;
    cudaError_t e = ensure_smem_attr((const void *)kern, configured, FUSED_SMEM_BYTES);
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
