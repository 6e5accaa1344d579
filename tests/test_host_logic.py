"""Host logic of the library on the CPU (no GPU): the launch layout it derives from a message's lengths, the chunk plan
of the host-buffer pipeline, and a CPU MODEL of the kernels' GHASH regrouping.

The model follows DESIGN.md section 5.2 step by step -- virtual block sequence [pad | AAD | payload | length block] in
rows of 32, rows dealt to W warps balanced to +-1, per lane the recurrence Y <- Y.K xor X with K = H^32, one product
per lane with H^(1..32), one weight H^(blocks behind the run) per warp, XOR of everything, chunk chaining with
H^(blocks of the chunk) -- but does every field operation with the ORACLE's bit-serial multiply (oracle.gf_mul /
gf_pow), so it shares no arithmetic with the CUDA path; only the integers of the layout come from the library
(gcm_debug_row_layout / gcm_debug_plan_chunks).  It must equal the plain Horner chain of PAPER.md Eq. 1 (L191),
oracle.ghash, for every length and geometry: an off-by-one in the pad, the lane rotation of a ragged last row, a
warp weight or a chunk power fails here before any kernel runs ("CPU model of the GPU's power
bookkeeping vs step 7").
"""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def G():
    import paper_2602_23067_b200 as pkg
    return pkg


def xor(a: bytes, b: bytes) -> bytes:
    return bytes(x ^ y for x, y in zip(a, b))


ZERO = bytes(16)


def blocks_of(data: bytes):
    return [data[i: i + 16].ljust(16, b"\0") for i in range(0, len(data), 16)]


def model_launch(oracle, G, h: bytes, aad: bytes, c: bytes, warps: int, ctr_base: int = 0, last: bool = True,
                 final_len=None, final_aad_len=None):
    """GHASH contribution of one launch as the fused kernel regroups it; returns (sum, number of GHASH blocks)."""
    lay = G.gcm_debug_row_layout(len(c), len(aad), ctr_base, last, True)
    E, S, pad = lay["vblocks"], lay["rows"], lay["pad"]
    X = [ZERO] * pad + blocks_of(aad) + blocks_of(c)
    if last:
        fl = len(c) if final_len is None else final_len
        fa = len(aad) if final_aad_len is None else final_aad_len
        X.append((8 * fa).to_bytes(8, "big") + (8 * fl).to_bytes(8, "big"))
    assert len(X) == E and S == (E + 31) // 32 and lay["base"] == pad + lay["n_aad_blocks"]
    assert (lay["ctr_delta"] + lay["base"]) % (1 << 32) == (ctr_base + 2) % (1 << 32)      # counter of payload block 0
    assert lay["ctr_delta"] % 32 == 0                                                  # counter == virtual index mod 32
    K = oracle.gf_pow(h, 32)
    total = ZERO
    for w in range(warps):
        r0, r1 = (w * S) // warps, ((w + 1) * S) // warps
        if r0 == r1:
            continue
        rem = E - 32 * (S - 1) if r1 == S else 32
        warp_sum = ZERO
        for lane in range(32):
            Y = ZERO
            for row in range(r0, r1):
                v = 32 * row + lane
                if v < E:
                    Y = xor(oracle.gf_mul(Y, K), X[v])
            e = ((rem - lane - 1) & 31) + 1
            warp_sum = xor(warp_sum, oracle.gf_mul(Y, oracle.gf_pow(h, e)))
        behind = E - 32 * r1 if r1 < S else 0
        total = xor(total, oracle.gf_mul(warp_sum, oracle.gf_pow(h, behind)))
    return total, E - pad


def test_row_layout_invariants(G):
    rng = np.random.default_rng(7100)
    cases = [(0, 0), (1, 0), (15, 3), (16, 16), (17, 0), (512, 0), (513, 2880), (16 * 32 * 7 + 5, 17), (1 << 20, 2880),
             ((1 << 32) + 13, 777)] + [(int(rng.integers(0, 1 << 22)), int(rng.integers(0, 4000))) for _ in range(200)]
    for (n, a) in cases:
        for ctr_base in (0, 1 << 17, 12345 * 4096):
            lay = G.gcm_debug_row_layout(n, a, ctr_base, True, True)
            n_aad, n_blk, n_full = (a + 15) // 16, (n + 15) // 16, n // 16
            assert 0 <= lay["pad"] < 32 and lay["n_aad_blocks"] == n_aad
            assert lay["vblocks"] == lay["pad"] + n_aad + n_blk + 1 and lay["rows"] == (lay["vblocks"] + 31) // 32
            assert (lay["base"] + lay["ctr_delta"]) % (1 << 32) == (ctr_base + 2) % (1 << 32) and lay["ctr_delta"] % 32 == 0
            # fast rows hold nothing but whole payload blocks
            assert 32 * lay["fast_lo"] >= lay["base"] or lay["fast_lo"] == lay["fast_hi"]
            assert 32 * lay["fast_hi"] <= lay["base"] + n_full or lay["fast_lo"] == lay["fast_hi"]
            assert lay["fast_hi"] >= lay["fast_lo"]
        un = G.gcm_debug_row_layout(n, a, 0, True, False)
        assert un["fast_lo"] == un["fast_hi"] == 0                                 # unaligned buffers: byte-granular path only
        mid = G.gcm_debug_row_layout(n, a, 0, False, True)
        assert mid["len_block"] == 0 and mid["vblocks"] == mid["pad"] + (a + 15) // 16 + (n + 15) // 16
    assert G.gcm._L.gcm_debug_row_layout((1 << 36) - 31, 0, 0, 1, 1, None) == G.GCM_ERR_ARG
    import ctypes
    out = G.gcm.GcmRowLayout()
    assert G.gcm._L.gcm_debug_row_layout((1 << 36) - 31, 0, 0, 1, 1, ctypes.byref(out)) == G.GCM_ERR_LEN


def test_model_of_the_kernel_regrouping_equals_horner(G, oracle):
    """Every total block count 1..75 (all lane rotations of the ragged last row, one to three rows) under several
    warp counts, then larger ragged messages."""
    rng = np.random.default_rng(7200)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    for n in list(range(0, 16 * 75, 16 * 3 + 5)) + [0, 1, 15, 16, 17, 511, 512, 513]:
        for a in (0, 7, 16, 100):
            aad = rng.integers(0, 256, a, dtype=np.uint8).tobytes()
            c = rng.integers(0, 256, n, dtype=np.uint8).tobytes()
            ref = oracle.ghash(h, aad, c)
            for warps in (1, 2, 3, 16):
                got, _ = model_launch(oracle, G, h, aad, c, warps)
                assert got == ref, (n, a, warps)
    for (n, a, warps) in [(16 * 32 * 9 + 16 * 5 + 3, 2880, 7), (16 * 32 * 20, 0, 32), (16 * 32 * 4 + 1, 45, 5)]:
        aad = rng.integers(0, 256, a, dtype=np.uint8).tobytes()
        c = rng.integers(0, 256, n, dtype=np.uint8).tobytes()
        assert model_launch(oracle, G, h, aad, c, warps)[0] == oracle.ghash(h, aad, c), (n, a, warps)


def test_model_of_the_chunk_chain_equals_horner(G, oracle):
    """The host pipeline: chunk k covers payload blocks [off/16, ...) with its own launch layout, the running state is
    Y_k = Y_(k-1) . H^(GHASH blocks of chunk k) xor S_k, the AAD rides with the first chunk and the length block with
    the last.  Cuts chosen by hand here (multiples of 16), the library's own plan is checked below."""
    rng = np.random.default_rng(7300)
    h = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
    for cuts, a in [([16 * 40, 16 * 7, 16 * 33 + 9], 45), ([16 * 32, 16 * 32], 0), ([16, 16, 16, 5], 2880), ([16 * 100, 0 + 16 * 3 - 2], 16)]:
        aad = rng.integers(0, 256, a, dtype=np.uint8).tobytes()
        c = rng.integers(0, 256, sum(cuts), dtype=np.uint8).tobytes()
        Y, off = ZERO, 0
        for k, n in enumerate(cuts):
            last = k == len(cuts) - 1
            s_k, n_k = model_launch(oracle, G, h, aad if k == 0 else b"", c[off: off + n], 3, ctr_base=off // 16, last=last,
                                    final_len=len(c), final_aad_len=len(aad))
            Y = xor(oracle.gf_mul(Y, oracle.gf_pow(h, n_k)), s_k) if k else s_k
            off += n
        assert Y == oracle.ghash(h, aad, c), cuts


def test_chunk_plan_invariants(G):
    MiB = 1 << 20
    rng = np.random.default_rng(7400)
    lens = [0, 1, 15, 2 * MiB - 1, 2 * MiB, 2 * MiB + 1, 17 * MiB, 64 * MiB, 64 * MiB + 12345, 201 * MiB, 577 * MiB + 3,
            4 << 30, (1 << 36) - 32] + [int(rng.integers(1, 1 << 33)) for _ in range(200)]
    for n in lens:
        plan = G.gcm_debug_plan_chunks(n)
        assert sum(plan) == n and len(plan) >= 1
        assert all(p % (2 * MiB) == 0 and p > 0 for p in plan[:-1]), n       # every cut on a 2 MiB (so 16-byte) boundary
        assert max(plan) <= 64 * MiB and (plan[-1] > 0 or n == 0) and plan[-1] <= 2 * MiB
        assert plan[0] <= 2 * MiB                                            # first upload, last download: not overlapped
        # small chunks at both ends, growing inwards (the chunk where the two ramps meet takes what is left)
        if len(plan) >= 8:
            assert plan[0] <= plan[1] <= plan[2] and plan[-1] <= plan[-2] <= plan[-3], (n, plan[:4], plan[-4:])
        assert len(plan) <= 1100
    assert len(G.gcm_debug_plan_chunks(64 * MiB)) <= 10                      # few chunks: a copy costs ~30 us on top of its bytes


# ---- CPU model of the tensor-core GHASH: GF(2) matrix products as integer counts + parity ----------
def _bits_mem(block: bytes) -> np.ndarray:
    """The 128 bits of a block in the kernels' "mem" order: bit b of little-endian word i is index 32 i + b."""
    w = np.frombuffer(block, dtype="<u4")
    return ((w[:, None] >> np.arange(32, dtype=np.uint32)[None, :]) & 1).astype(np.int64).reshape(128)


def _block_of_bits(bits: np.ndarray) -> bytes:
    w = (bits.reshape(4, 32).astype(np.uint64) << np.arange(32, dtype=np.uint64)[None, :]).sum(axis=1).astype("<u4")
    return w.tobytes()


def _matrix_of(oracle, p: bytes) -> np.ndarray:
    """M(P): row k = the bits of (unit block k) . P, by the oracle's bit-serial multiply."""
    m = np.zeros((128, 128), dtype=np.int64)
    for k in range(128):
        u = np.zeros(128, dtype=np.int64)
        u[k] = 1
        m[k] = _bits_mem(oracle.gf_mul(_block_of_bits(u), p))
    return m


def test_model_of_the_tensor_ghash_equals_horner(oracle):
    """What gcm_ghash_tc_kernel computes, with the ORACLE's field operations and plain integer arithmetic in place of the
    tensor core: the virtual sequence [pad | AAD | C | length block] in whole chunks of 16 slices of 128 consecutive
    blocks; per chunk and row j the COUNT sum_t bits(X_(128 t + j)) x M(K^(15 - t)) over the integers with the operand
    nibbles weighted 0.5 / 1 / 2 / 2 and the matrix rows 2 / 1 / 0.5 / 0.5 (every product exactly 1), its parity as Z_j,
    Y_j <- Y_j . K^16 xor Z_j, at the end sum_j Y_j . H^(128 - j) and the weight of the chunks behind the run.  Two CTAs
    with different numbers of chunks.  Must equal the Horner chain of PAPER.md Eq. 1 (L191): a wrong matrix
    orientation, bit order, weight pairing, slice power or row exponent fails here without a GPU."""
    rng = np.random.default_rng(31337)
    key = rng.integers(0, 256, 32, dtype=np.uint8).tobytes()
    h = oracle.hash_subkey(key)
    K = oracle.gf_pow(h, 128)
    L, SL = 16, 128
    mats = [_matrix_of(oracle, oracle.gf_pow(h, 128 * e)) for e in range(L)]
    # e2m1 values of the operand nibbles for message bit positions 4m + j, j = 0..3, and of the matrix rows that meet them
    a_w = np.tile(np.array([0.5, 1.0, 2.0, 2.0]), 32)
    b_w = np.tile(np.array([2.0, 1.0, 0.5, 0.5]), 32)
    for (n, a) in ((3 * 32768 + 5, 33), (2 * 32768 - 16 * 3, 0)):
        aad, c = rng.integers(0, 256, a, dtype=np.uint8).tobytes(), rng.integers(0, 256, n, dtype=np.uint8).tobytes()
        lenblk = (8 * a).to_bytes(8, "big") + (8 * n).to_bytes(8, "big")
        real = blocks_of(aad) + blocks_of(c) + [lenblk]
        nchunks = (len(real) + L * SL - 1) // (L * SL)
        X = [ZERO] * (nchunks * L * SL - len(real)) + real                 # leading zero blocks are free
        total = ZERO
        cuts = [0, nchunks // 2, nchunks] if nchunks > 1 else [0, nchunks]
        for c0, c1 in zip(cuts[:-1], cuts[1:]):                             # one "CTA" per run of chunks
            Y = [ZERO] * SL
            for ch in range(c0, c1):
                counts = np.zeros((SL, 128))
                for t in range(L):
                    rows = np.stack([_bits_mem(X[(ch * L + t) * SL + j]) for j in range(SL)]).astype(np.float64)
                    counts += (rows * a_w[None, :]) @ (mats[L - 1 - t] * b_w[:, None])
                assert np.all(counts == np.floor(counts)) and counts.max() < 2 ** 24
                Z = [_block_of_bits((counts[j].astype(np.int64) & 1)) for j in range(SL)]
                KL = oracle.gf_pow(h, 128 * L)
                Y = [xor(oracle.gf_mul(Y[j], KL), Z[j]) for j in range(SL)]
            part = ZERO
            for j in range(SL):
                part = xor(part, oracle.gf_mul(Y[j], oracle.gf_pow(h, 128 - j)))
            behind = (nchunks - c1) * L * SL
            if behind:
                part = oracle.gf_mul(part, oracle.gf_pow(h, behind))
            total = xor(total, part)
        assert total == oracle.ghash(h, aad, c), (n, a)
    assert K == oracle.gf_pow(oracle.gf_pow(h, 64), 2)
