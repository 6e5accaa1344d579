// gcm_fused.cu -- the hot path: SURVEY.md 8(a) steps a3-a11 in ONE kernel.
//
//   AES-CTR keystream (a4, a5) -> XOR into the payload (a6) -> GHASH of the ciphertext while it is
//   still in registers (a7) -> per-thread / warp / CTA / cross-CTA combination with precomputed
//   powers of H (a8, a9) -> AAD + length block, E_K(J0), tag,
//   constant-time compare (a10, a11).
//
// What differs from the paper's kernels (prior art for Ampere/Ada/Hopper):
//   * one fused pass instead of an AES-CTR kernel followed by a GHASH kernel (the ciphertext never
//     crosses HBM twice);
//   * the "tree" is flattened.  The virtual block sequence [pad | AAD | payload] is cut into rows of
//     32 blocks; a warp owns a contiguous run of rows and lane l of the warp the l-th block of each.
//     Every lane therefore runs the SAME recurrence  Y <- Y.K xor X  with the one fixed multiplier
//     K = H^32 (independent of the launch geometry and of the message), and is corrected once by
//     H^(1..32), the warp by H^(blocks behind the warp's run), and the partials are XORed by the
//     last CTA to finish.  The sum is the paper's sum of X_i . H^(N-i+1); only the association
//     differs, and the field is exact, so the bits are identical;
//   * the multiply by the fixed K is an 8-bit Shoup table in shared memory (conflict-free by lane
//     rotation), AES rounds are T-tables replicated per lane (conflict-free, constant-time).  On
//     sm_100a the binding unit is the shared-memory pipe;
//   * counters of a lane's consecutive blocks differ by 32, so for 8 rows at a time only the low
//     counter byte changes: of rounds 1 and 2 only 1 + 4 table reads depend on it, the other 3 + 12
//     are cached per lane and refreshed every 8th row (in addition to the 12 round-1 reads of the
//     constant IV columns, done once per thread).
//
// Counter block of payload block g is IV || BE32(g + 2): a function of g only.
#include "gcm_common.cuh"
#include "gf128.cuh"
#include "gcm_fused.cuh"

#include "gcm_device.cuh"

// H^d for d < 2^36 from the radix-512 digit table: four factors, two multiply levels, every lane
// of the warp takes part (lane & 3 picks the digit) and ends up with the product.
__device__ __forceinline__ uint4 warp_h_power(const uint4 *hx, uint64_t d, uint32_t lane, uint64_t d_max)
{
    const uint32_t k = lane & 3;
    const uint32_t digit = (uint32_t)(d >> (HX_RADIX_BITS * k)) & ((1u << HX_RADIX_BITS) - 1);
    uint4 f = __ldg(hx + (k << HX_RADIX_BITS) + digit);
    // d_max (launch-uniform bound on d) says how many digits can be non-zero: short messages skip levels
    const int levels = d_max < (1ull << HX_RADIX_BITS) ? 0 : (d_max < (1ull << (2 * HX_RADIX_BITS)) ? 1 : 2);
    for (int o = 1; o <= levels; o++) {
        const int m = 1 << (o - 1);
        uint4 g;
        g.x = __shfl_xor_sync(0xFFFFFFFFu, f.x, m); g.y = __shfl_xor_sync(0xFFFFFFFFu, f.y, m);
        g.z = __shfl_xor_sync(0xFFFFFFFFu, f.z, m); g.w = __shfl_xor_sync(0xFFFFFFFFu, f.w, m);
        f = gf_mul_mem(f, g);
    }
    // lanes with k = 0 hold the product of the digits that can be non-zero; hand it to every lane
    f.x = __shfl_sync(0xFFFFFFFFu, f.x, lane & ~3u); f.y = __shfl_sync(0xFFFFFFFFu, f.y, lane & ~3u);
    f.z = __shfl_sync(0xFFFFFFFFu, f.z, lane & ~3u); f.w = __shfl_sync(0xFFFFFFFFu, f.w, lane & ~3u);
    return f;
}

template <int NR, int MODE, int TPB>
__global__ void __launch_bounds__(TPB, 1)
gcm_fused_kernel(const __grid_constant__ GcmParams p)
{
    extern __shared__ __align__(1024) uint8_t sm[];
    __shared__ bool s_last;
    __shared__ uint4 s_ekj0;
    const uint32_t t = threadIdx.x, lane = t & 31, lane4 = lane * 4;
    // broadcast from lane 0: tells the compiler the warp index (and the row loop below) is warp-uniform,
    // so the shared-memory base stays in a uniform register and folds into every LDS address
    const uint32_t warp = __shfl_sync(0xFFFFFFFFu, t >> 5, 0);
    uint4 *red = reinterpret_cast<uint4 *>(sm + RED_OFF);

    // this warp's run of rows (a8: geometry-agnostic, the result does not depend on it)
    const uint32_t S = p.rows, Q = p.rows_per_warp;
    const uint64_t wg = (uint64_t)blockIdx.x * (TPB / 32) + warp;
    const uint64_t r0_64 = wg * Q;
    const uint32_t r0 = r0_64 < S ? (uint32_t)r0_64 : S;
    const uint32_t r1 = (uint64_t)r0 + Q < S ? r0 + Q : S;
    const bool has_rows = r0 < r1;

    {
        KtabRegs<TPB> kr;
        ktab_load<TPB>(kr, p.tab.ktab);
        if (MODE != MODE_GHASH) fill_aes_tables<TPB>(sm, p.tab.te0);
        ktab_store<TPB>(kr, sm);
    }
    const bool tail_warp = has_rows && r1 == S;          // owns the last (possibly ragged) row
    __syncthreads();

    uint32_t sel[8];
#pragma unroll
    for (int r = 0; r < 8; r++) sel[r] = ((lane + r) & 7) << 4;
    CtrConst cc = {0, 0, 0, 0};
    CtrCache cu = {0, 0, 0, 0};
    if (MODE != MODE_GHASH) {
        cc = ctr_const(p.rk, p.iv[0], p.iv[1], p.iv[2], sm, lane4);
        // a3: E_K(J0), J0 = IV || 0^31 || 1, by the last warp of every CTA while the others start their rows
        // (any CTA may turn out to be the finisher); it reaches the finishing thread through shared memory
        if (warp == TPB / 32 - 1) {
            const CtrCache c1 = ctr_cache(p.rk, sm, lane4, cc, 1u);
            const uint4 ek = aes_ctr_block<NR>(p.rk, sm, lane4, cc, c1, 1u);
            if (lane == 0) s_ekj0 = ek;
        }
    }

    uint4 Y = make_uint4(0, 0, 0, 0);
    uint4 pre = make_uint4(0, 0, 0, 0);
    bool have_pre = false;

    // a8, first half: the weight each lane's partial is multiplied by at the end of the run,
    //     V_l = H^(blocks from the lane's last block to the end of the run) . H^(blocks behind the run).
    // In the ragged last row only lanes < rem folded a block; rotating the lane order by rem keeps the first
    // exponent in 1..32.  The generic products behind V (up to three per warp) are NOT done before the rows or
    // after them, where all warps of the SM would do them at once with the table pipe idle, but in the middle
    // of the run, at a row that differs from warp to warp: the other warps keep the shared-memory pipe busy.
    uint4 V = make_uint4(0, 0, 0, 0);
    const uint32_t rmid = r0 + (uint32_t)(((uint64_t)(r1 - r0) * (warp + 1)) / (TPB / 32 + 1));

    for (uint32_t row = r0; row < r1; row++) {
        if (row == rmid) {                               // once per run, at a warp-specific row (see above)
            const uint32_t rem = tail_warp ? (uint32_t)(p.vblocks - 32ull * (S - 1)) : 32u;   // 1..32
            V = __ldg(p.tab.hpow + (((rem - lane - 1) & 31) + 1));
            if (!tail_warp) V = gf_mul_mem(V, warp_h_power(p.tab.hx, p.vblocks - 32ull * r1, lane, p.vblocks));
        }
        const uint64_t v = 32ull * row + lane;          // virtual block index
        const bool fast = row >= p.fast_lo && row < p.fast_hi;
        uint4 x = make_uint4(0, 0, 0, 0);
        uint32_t cbytes = 0;                            // payload bytes in this block (0: pad / AAD / beyond the end)
        uint64_t g = 0;                                 // payload block index
        bool valid = true;
        if (fast) {
            g = v - p.base;
            x = have_pre ? pre : ld16_stream(p.in + 16 * g);
            cbytes = 16;
            have_pre = row + 1 < r1 && row + 1 < p.fast_hi;
            if (have_pre) pre = ld16_stream(p.in + 16 * g + 512);
        } else {
            have_pre = false;
            valid = v < p.vblocks;
            if (valid && v >= p.pad) {
                const uint64_t u = v - p.pad;
                if (u < p.n_aad_blocks) {
                    const uint64_t rem = p.aad_len - 16 * u;
                    x = load_bytes(p.aad + 16 * u, rem < 16 ? (uint32_t)rem : 16u);
                } else {
                    g = u - p.n_aad_blocks;
                    const uint64_t rem = p.len - 16 * g;
                    cbytes = rem < 16 ? (uint32_t)rem : 16u;
                    x = (cbytes == 16 && p.aligned) ? ld16_stream(p.in + 16 * g) : load_bytes(p.in + 16 * g, cbytes);
                }
            }
        }
        // a7: multiply the running value by K; independent of this row's AES, so they interleave
        const uint4 ym = ghash_mul_k(sm, sel, Y);
        uint4 X = x;
        if (MODE != MODE_GHASH) {
            // a4: counter from the virtual index alone; the upper 24 bits are warp-uniform and change
            // every 8th row, when rounds 1-2 are re-cached
            const uint32_t ctr = (uint32_t)v + p.ctr_delta;
            if (row == r0 || (ctr & 0xE0u) == 0) cu = ctr_cache(p.rk, sm, lane4, cc, ctr);
            const uint4 ks = aes_ctr_block<NR>(p.rk, sm, lane4, cc, cu, ctr);     // a5
            const uint4 y = xor4(x, ks);                                   // a6
            if (cbytes == 16 && (fast || p.aligned)) st16_stream(p.out + 16 * g, y);
            else if (cbytes) store_bytes(p.out + 16 * g, y, cbytes);
            if (MODE == MODE_ENCRYPT && cbytes) X = keep_bytes(y, cbytes);
        }
        if (fast || valid) Y = xor4(ym, X);
    }
    // a8, second half: one product per lane, XOR over the warp, XOR over the CTA
    uint4 part = make_uint4(0, 0, 0, 0);
    if (has_rows) part = gf_mul_mem(Y, V);
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        part.x ^= __shfl_xor_sync(0xFFFFFFFFu, part.x, o); part.y ^= __shfl_xor_sync(0xFFFFFFFFu, part.y, o);
        part.z ^= __shfl_xor_sync(0xFFFFFFFFu, part.z, o); part.w ^= __shfl_xor_sync(0xFFFFFFFFu, part.w, o);
    }
    if (lane == 0) red[warp] = part;
    __syncthreads();
    if (warp == 0) {
        part = lane < TPB / 32 ? red[lane] : make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) {
            part.x ^= __shfl_xor_sync(0xFFFFFFFFu, part.x, o); part.y ^= __shfl_xor_sync(0xFFFFFFFFu, part.y, o);
            part.z ^= __shfl_xor_sync(0xFFFFFFFFu, part.z, o); part.w ^= __shfl_xor_sync(0xFFFFFFFFu, part.w, o);
        }
    }
    // a9: last-CTA-done combination of the partials
    if (t == 0) {
        p.partials[blockIdx.x] = part;
        __threadfence();
        const unsigned ticket = atomicAdd(p.counter, 1u);
        s_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    uint4 acc = make_uint4(0, 0, 0, 0);
    for (uint32_t j = t; j < gridDim.x; j += TPB) acc = xor4(acc, __ldcg(p.partials + j));
    acc = cta_xor_reduce(acc, red);
    if (t == 0) {
        if (p.chain_in != nullptr) acc = xor4(acc, gf_mul_mem(*p.chain_in, *p.chain_pow));
        if (p.chain_out != nullptr) {       // a middle chunk of a longer message: hand the state on
            *p.chain_out = acc;
            *p.counter = 0;
            return;
        }
        // a10: length block BE64(8a) || BE64(8 len), one more multiply by H
        const uint64_t abits = p.final_aad_len * 8, cbits = p.final_len * 8;
        const uint4 L = make_uint4(bswap32((uint32_t)(abits >> 32)), bswap32((uint32_t)abits),
                                   bswap32((uint32_t)(cbits >> 32)), bswap32((uint32_t)cbits));
        const uint4 Sg = gf_mul_mem(xor4(acc, L), __ldg(p.tab.h));
        if (MODE == MODE_GHASH) {
            *p.tag_out = Sg;
        } else {
            // a11: tag = E_K(J0) xor S; constant-time compare
            const uint4 tag = xor4(Sg, s_ekj0);
            if (MODE == MODE_ENCRYPT) {
                *p.tag_out = tag;
            } else {
                uint4 expect = make_uint4(p.tag_expect[0], p.tag_expect[1], p.tag_expect[2], p.tag_expect[3]);
                if (p.tag_in != nullptr) expect = *p.tag_in;
                const uint32_t diff = (tag.x ^ expect.x) | (tag.y ^ expect.y) | (tag.z ^ expect.z) | (tag.w ^ expect.w);
                *p.status = diff != 0 ? 1 : 0;
            }
        }
        *p.counter = 0;   // ready for the next launch on this context
    }
}

// ---- host side ------------------------------------------------------------------------------------
template <int NR, int MODE, int TPB>
static cudaError_t launch_one(int blocks, const GcmParams &p, cudaStream_t s)
{
    static bool configured[64] = {false};   // per instantiation and device; the attribute is sticky
    auto kern = gcm_fused_kernel<NR, MODE, TPB>;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, FUSED_SMEM_BYTES);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    kern<<<blocks, TPB, FUSED_SMEM_BYTES, s>>>(p);
    return cudaGetLastError();
}

template <int TPB>
static cudaError_t launch_tpb(int nr, int mode, int blocks, const GcmParams &p, cudaStream_t s)
{
    if (mode == MODE_GHASH) return launch_one<10, MODE_GHASH, TPB>(blocks, p, s);
    if (nr == 10) return mode == MODE_ENCRYPT ? launch_one<10, MODE_ENCRYPT, TPB>(blocks, p, s)
                                              : launch_one<10, MODE_DECRYPT, TPB>(blocks, p, s);
    return mode == MODE_ENCRYPT ? launch_one<14, MODE_ENCRYPT, TPB>(blocks, p, s)
                                : launch_one<14, MODE_DECRYPT, TPB>(blocks, p, s);
}

cudaError_t launch_fused(int nr, int mode, int threads, int blocks, const GcmParams &p, cudaStream_t s)
{
    if (threads == 256) return launch_tpb<256>(nr, mode, blocks, p, s);
    if (threads == 384) return launch_tpb<384>(nr, mode, blocks, p, s);
    return launch_tpb<512>(nr, mode, blocks, p, s);
}
