"""GPU parity for GHASH on the tensor cores (gcm_set_ghash_engine; csrc/gcm_tc.cu and csrc/gcm_ghash_tc.cu).

The multiply by a power of H is done as a GF(2) matrix-vector product on tcgen05.mma (0/1 operands as e2m1, counts in
fp32, parity); Eq. 1 leaves the method of the multiply open (reading S7), so the result
must be THE GHASH value: every ciphertext byte and every tag / GHASH byte is compared with the oracle (integer work,
bit-exact).  Shapes are chosen around what the kernels treat specially: chunks of TC_L = 8 rows per lane, runs that are
one row short, the ragged last row that stays off the tensor core, the 32 KiB chunks and the 4 MiB threshold of the
GHASH-only kernel, grids smaller and larger than the number of chunks.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

THREADS = os.cpu_count() or 1


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2602_23067_b200 as pkg
    return pkg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rnd(rng, n):
    return rng.integers(0, 256, n, dtype=np.uint8)


def oracle_encrypt(oracle, key, iv, aad, pt):
    if len(pt) <= 1 << 16:
        ct, tag = oracle.gcm_encrypt(key, iv, aad, pt)
        return np.asarray(ct, dtype=np.uint8), bytes(tag)
    ct, tag = oracle.gcm_encrypt_threaded(key, iv, aad, pt, THREADS, 1 << 16)
    return np.asarray(ct, dtype=np.uint8), bytes(tag)


def test_engine_selector(G):
    ctx = G.gcm_init(bytes(16))
    try:
        assert G.gcm_get_ghash_engine(ctx) == G.GCM_GHASH_AUTO
        for e in (G.GCM_GHASH_TABLE, G.GCM_GHASH_TENSOR, G.GCM_GHASH_AUTO):
            G.gcm_set_ghash_engine(ctx, e)
            assert G.gcm_get_ghash_engine(ctx) == e
        with pytest.raises(G.GcmError):
            G.gcm_set_ghash_engine(ctx, 3)
    finally:
        G.gcm_destroy(ctx)


@pytest.mark.parametrize("grid", [0, 1, 7])
def test_tensor_engine_encrypt_decrypt_shapes(G, oracle, grid):
    """gcm_tc_kernel for AES-128 and AES-256, encrypt and decrypt: empty / tiny / ragged messages, one to many chunks
    of 8 rows per lane, AAD of 0 .. 2880 bytes, unaligned and in-place buffers; with one CTA (every warp runs many
    chunks), seven and one per SM.  Then a flipped ciphertext bit, a flipped AAD bit and a wrong tag: refused, zeros."""
    rng = np.random.default_rng(9960 + grid)
    per_cta = 12 * 512                                        # bytes of one row of every producer warp of a CTA
    lens = [0, 1, 15, 16, 17, 511, 512, 513, per_cta - 32, per_cta, 3 * per_cta + 5, 8 * per_cta - 32, 8 * per_cta + 16,
            9 * per_cta - 33, 17 * per_cta + 4097, (1 << 20) + 13]
    if grid == 0:
        lens += [3 << 20, (5 << 20) + 511]
    for klen in (16, 32):
        key = rnd(rng, klen).tobytes()
        ctx = G.gcm_init(key)
        try:
            G.gcm_set_geometry(ctx, grid, 0)
            G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)
            for i, n in enumerate(lens):
                a = [0, 1, 16, 17, 100, 2880][i % 6]
                iv, aad, pt = rnd(rng, 12).tobytes(), rnd(rng, a), rnd(rng, n)
                want_ct, want_tag = oracle_encrypt(oracle, key, iv, aad, pt)
                off = 5 if i % 4 == 3 else 0                   # every fourth message unaligned
                big_in = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
                big_in[off: off + n] = dev(pt)
                in_place = i % 5 == 2
                big_out = big_in if in_place else torch.full((n + 64,), 0xEE, dtype=torch.uint8, device="cuda")
                d_aad = dev(aad) if a else None
                tag = G.gcm_encrypt(ctx, iv, d_aad, big_in[off: off + n], big_out[off: off + n])
                got = big_out[off: off + n].cpu().numpy()
                assert np.array_equal(got, want_ct), (klen, n, a, "ciphertext")
                assert bytes(tag) == want_tag, (klen, n, a, "tag")
                if not in_place:                               # nothing written outside the message
                    assert int(big_out[:off].cpu().numpy().astype(np.int64).sum()) == 0xEE * off
                    assert bool((big_out[off + n:] == 0xEE).all())
                # decrypt from oracle-written ciphertext
                d_ct = dev(want_ct) if n else torch.zeros(0, dtype=torch.uint8, device="cuda")
                d_pt = torch.full((n,), 0xEE, dtype=torch.uint8, device="cuda")
                assert G.gcm_decrypt_verify(ctx, iv, d_aad, d_ct, d_pt, want_tag) == G.GCM_OK
                assert np.array_equal(d_pt.cpu().numpy(), pt), (klen, n, a, "plaintext")
                # forgeries
                bad_tag = bytes([want_tag[0] ^ 1]) + want_tag[1:]
                assert G.gcm_decrypt_verify(ctx, iv, d_aad, d_ct, d_pt, bad_tag) == G.GCM_ERR_AUTH
                assert not bool(d_pt.any())
                if n:
                    forged = want_ct.copy()
                    forged[int(rng.integers(0, n))] ^= 0x10
                    d_pt.fill_(0xEE)
                    assert G.gcm_decrypt_verify(ctx, iv, d_aad, dev(forged), d_pt, want_tag) == G.GCM_ERR_AUTH
                    assert not bool(d_pt.any())
                if a:
                    aad2 = aad.copy()
                    aad2[a - 1] ^= 0x80
                    d_pt.fill_(0xEE)
                    assert G.gcm_decrypt_verify(ctx, iv, dev(aad2), d_ct, d_pt, want_tag) == G.GCM_ERR_AUTH
                    assert not bool(d_pt.any())
        finally:
            G.gcm_destroy(ctx)


def test_tensor_engine_equals_table_engine_at_64_mib(G, oracle):
    """64 MiB + 5 bytes, AES-256: 74 rows per lane = ten chunks with the running value fed back nine times; the
    ciphertext byte for byte against the oracle (and of both engines against each other), the tag against the
    oracle's segment identity (pinned against OpenSSL at this size in tests/test_oracle_full_size.py)."""
    import workloads
    rng = np.random.default_rng(9970)
    key, iv, aad = rnd(rng, 32).tobytes(), rnd(rng, 12).tobytes(), rnd(rng, 2880)
    n = (64 << 20) + 5
    pt = workloads.random_payload(rng, n)
    d_pt = dev(pt)
    ctx = G.gcm_init(key)
    try:
        outs = []
        for e in (G.GCM_GHASH_TABLE, G.GCM_GHASH_TENSOR):
            G.gcm_set_ghash_engine(ctx, e)
            d_ct = torch.empty_like(d_pt)
            outs.append((d_ct, G.gcm_encrypt(ctx, iv, dev(aad), d_pt, d_ct)))
        assert torch.equal(outs[0][0], outs[1][0])
        ct = outs[1][0].cpu().numpy()
        h = oracle.hash_subkey(key)
        s = oracle.ghash_segmented(h, aad, ct, 1 << 16, THREADS)
        want_tag = bytes(x ^ y for x, y in zip(s, oracle.ek_j0(key, iv)))
        assert bytes(outs[0][1]) == want_tag and bytes(outs[1][1]) == want_tag
        assert np.array_equal(oracle.ctr_xor(key, iv, pt, threads=THREADS), ct)      # every ciphertext byte
    finally:
        G.gcm_destroy(ctx)


@pytest.mark.parametrize("grid", [0, 3, 200])
def test_tc2_chain_shapes(G, oracle, grid):
    """gcm_tc2_kernel (AES warps + tensor-core GHASH warps) between the two row-kernel links, engine TENSOR: lengths on
    and around the 8 MiB threshold and around whole 128-block slices behind the 254-block head (0, 1, 127 blocks and a
    ragged byte count left for the last link), one to many chunks of 7 slices per CTA (3 CTAs: hundreds of chunks each;
    200 CTAs: more CTAs than the SMs), AAD 0 / 16 / 2880, both key sizes, in place.  Every ciphertext byte and the tag
    against the oracle; decrypt from oracle-written ciphertext; a forged byte inside the tensor stretch, one in the head
    and one in the tail: refused and zero-filled."""
    import workloads
    rng = np.random.default_rng(9995 + grid)
    M = 8 << 20
    head = 254 * 16
    lens = [M, M + 1, M - 16 + head % 2048, head + 2048 * 4096, head + 2048 * 4096 + 2047, head + 2048 * 4099 + 16 * 127 + 5, 3 * M + 777]
    for klen in (16, 32):
        key = rnd(rng, klen).tobytes()
        ctx = G.gcm_init(key)
        try:
            G.gcm_set_geometry(ctx, grid, 0)
            G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)
            for i, n in enumerate(lens):
                a = [0, 16, 2880][i % 3]
                iv, aad, pt = rnd(rng, 12).tobytes(), rnd(rng, a), workloads.random_payload(rng, n)
                want_ct, want_tag = oracle_encrypt(oracle, key, iv, aad, pt)
                d_aad = dev(aad) if a else None
                d_in = dev(pt)
                d_out = d_in if i % 3 == 1 else torch.full((n,), 0xEE, dtype=torch.uint8, device="cuda")
                tag = G.gcm_encrypt(ctx, iv, d_aad, d_in, d_out)
                assert np.array_equal(d_out.cpu().numpy(), want_ct), (klen, n, a, "ciphertext")
                assert bytes(tag) == want_tag, (klen, n, a, "tag")
                d_ct = dev(want_ct)
                d_pt = torch.full((n,), 0xEE, dtype=torch.uint8, device="cuda")
                assert G.gcm_decrypt_verify(ctx, iv, d_aad, d_ct, d_pt, want_tag) == G.GCM_OK
                assert np.array_equal(d_pt.cpu().numpy(), pt), (klen, n, a, "plaintext")
                for pos in (7, head + 2048 * 1000 + 3, n - 1):
                    forged = want_ct.copy()
                    forged[pos] ^= 0x04
                    d_pt.fill_(0xEE)
                    assert G.gcm_decrypt_verify(ctx, iv, d_aad, dev(forged), d_pt, want_tag) == G.GCM_ERR_AUTH, (n, pos)
                    assert not bool(d_pt.any())
            # the asynchronous forms: device tag, device verdict word
            n = lens[-1]
            iv, aad, pt = rnd(rng, 12).tobytes(), rnd(rng, 33), workloads.random_payload(rng, n)
            want_ct, want_tag = oracle_encrypt(oracle, key, iv, aad, pt)
            d_tag = torch.zeros(16, dtype=torch.uint8, device="cuda")
            d_ct = torch.empty(n, dtype=torch.uint8, device="cuda")
            G.gcm_encrypt_async(ctx, iv, dev(aad), dev(pt), d_ct, d_tag)
            torch.cuda.synchronize()
            assert d_tag.cpu().numpy().tobytes() == want_tag and np.array_equal(d_ct.cpu().numpy(), want_ct)
            d_status = torch.full((1,), 5, dtype=torch.int32, device="cuda")
            d_pt = torch.empty(n, dtype=torch.uint8, device="cuda")
            G.gcm_decrypt_verify_async(ctx, iv, dev(aad), d_ct, d_pt, d_tag, d_status)
            torch.cuda.synchronize()
            assert int(d_status.item()) == 0 and np.array_equal(d_pt.cpu().numpy(), pt)
            d_ct[n // 2] ^= 1
            G.gcm_decrypt_verify_async(ctx, iv, dev(aad), d_ct, d_pt, d_tag, d_status)
            torch.cuda.synchronize()
            assert int(d_status.item()) != 0 and not bool(d_pt.any())
        finally:
            G.gcm_destroy(ctx)


@pytest.mark.parametrize("engine", ["auto", "tensor"])
def test_ghash_stretch_kernel_shapes(G, oracle, engine):
    """gcm_ghash_async over at least 4 MiB (engine TENSOR) / 32 MiB (default engine) of aligned input: one launch of
    gcm_ghash_tc_kernel over [pad | AAD | C | length block] in whole 32 KiB chunks; the slices at both ends (pad, AAD, the
    first blocks of C; the ragged last block, the length block) are put together by hand, the rest by bulk copy.
    Lengths on and around the threshold and the chunk size, AAD 0 / 1 / 16 / 17 / 100 / 2880 bytes (AAD within one
    slice and across two), grids of 1, 5, 40, 148 and 300 CTAs (more CTAs than chunks included), both key sizes; one
    unaligned input, which must take the row kernel."""
    import workloads
    rng = np.random.default_rng(9980)
    M = 4 << 20
    cases = [(M, 0, 0), (M + 1, 16, 0), (M - 1, 2880, 0), (M + 32768, 1, 5), (M + 32767, 0, 1), (M + 32769, 17, 148),
             (5 * M + 12345, 2880, 300), (148 * 32768 * 2, 0, 0), (148 * 32768 * 2 + 32768 * 3 + 15, 100, 0), (3 * M, 16, 1)]
    if engine == "auto":        # the default engine takes the tensor path from 32 MiB on; below that the table kernel
        cases = [(8 * M, 0, 0), (8 * M - 1, 16, 0), (8 * M + 32769, 2880, 0), (25 * M + 7, 1, 40)]
    for klen in (16, 32):
        key = rnd(rng, klen).tobytes()
        h = oracle.hash_subkey(key)
        ctx = G.gcm_init(key)
        try:
            if engine == "tensor":
                G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)
            for (n, a, grid) in cases:
                G.gcm_set_geometry(ctx, grid, 0)
                aad, c = rnd(rng, a), workloads.random_payload(rng, n)
                want = oracle.ghash_segmented(h, aad, c, 1 << 16, THREADS)
                d_s = torch.full((16,), 0xEE, dtype=torch.uint8, device="cuda")
                G.gcm_ghash_async(ctx, dev(aad) if a else None, dev(c), d_s)
                torch.cuda.synchronize()
                assert d_s.cpu().numpy().tobytes() == want, (klen, n, a, grid)
            # the same bytes at an unaligned address
            G.gcm_set_geometry(ctx, 0, 0)
            n = M + 77
            c = workloads.random_payload(rng, n)
            big = torch.zeros(n + 32, dtype=torch.uint8, device="cuda")
            big[3: 3 + n] = dev(c)
            d_s = torch.zeros(16, dtype=torch.uint8, device="cuda")
            G.gcm_ghash_async(ctx, None, big[3: 3 + n], d_s)
            torch.cuda.synchronize()
            assert d_s.cpu().numpy().tobytes() == oracle.ghash_segmented(h, b"", c, 1 << 16, THREADS)
        finally:
            G.gcm_destroy(ctx)


def test_ghash_stretch_kernel_4_gib(G, oracle):
    """The bench shape of `--workload c5-ghash`: 4 GiB, 2880-byte AAD, default engine and geometry.  The oracle's
    weighted segments (ghash_segment, pinned at this size against OpenSSL in test_oracle_full_size.py), window by
    window as in test_gpu_full_configs.py."""
    from concurrent.futures import ThreadPoolExecutor
    rng = np.random.default_rng(9990)
    key, aad = rnd(rng, 32).tobytes(), rnd(rng, 2880)
    h = oracle.hash_subkey(key)
    n = 4 << 30
    gen = torch.Generator(device="cuda").manual_seed(1005)
    d_c = torch.randint(0, 256, (n,), dtype=torch.uint8, device="cuda", generator=gen)
    ctx = G.gcm_init(key)
    try:
        d_s = torch.zeros(16, dtype=torch.uint8, device="cuda")
        G.gcm_ghash_async(ctx, dev(aad), d_c, d_s)
        torch.cuda.synchronize()
        got = d_s.cpu().numpy().tobytes()
    finally:
        G.gcm_destroy(ctx)
    n_c, window, seg = n // 16, 256 << 20, 16 << 16
    acc = np.frombuffer(oracle.ghash_segment(h, aad, n_c + 1), np.uint8).copy()
    for off in range(0, n, window):
        c = d_c[off: off + window].cpu().numpy()
        jobs = [(c[s: s + seg], n_c - (off + s + seg) // 16 + 1) for s in range(0, window, seg)]
        with ThreadPoolExecutor(THREADS) as ex:
            for part in ex.map(lambda j: oracle.ghash_segment(h, j[0], j[1]), jobs):
                acc ^= np.frombuffer(part, np.uint8)
    lenblk = (8 * len(aad)).to_bytes(8, "big") + (8 * n).to_bytes(8, "big")
    acc ^= np.frombuffer(oracle.ghash_segment(h, lenblk, 0), np.uint8)
    assert got == acc.tobytes()


def test_tc2_chain_refuses_partial_overlap(G):
    """The links of the chain check only their own stretch; a partial overlap of the whole buffers (beyond the head
    link's 4064 bytes) must still be refused before anything is launched."""
    n = 16 << 20
    big = torch.zeros(n + (1 << 20), dtype=torch.uint8, device="cuda")
    ctx = G.gcm_init(bytes(32))
    try:
        G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)
        with pytest.raises(G.GcmError) as e:
            G.gcm_encrypt(ctx, bytes(12), None, big[:n], big[65536: 65536 + n])
        assert e.value.code == G.GCM_ERR_ARG
        assert not bool(big.any())
    finally:
        G.gcm_destroy(ctx)


@pytest.mark.parametrize("klen", [16, 32])
def test_default_engine_switches_at_its_threshold(G, oracle, klen):
    """GCM_GHASH_AUTO: an aligned message of exactly the threshold size (AES-128: 128 MiB, AES-256: 384 MiB) takes the
    gcm_tc2 chain, one block less the table kernel; both against the oracle (every ciphertext byte, the tag by the
    pinned segment identity), and the two ciphertexts agree on their common prefix."""
    import workloads
    rng = np.random.default_rng(9996 + klen)
    n = G.TC2_AUTO_BYTES[8 * klen]
    key, iv, aad = rnd(rng, klen).tobytes(), rnd(rng, 12).tobytes(), rnd(rng, 2880)
    pt = workloads.random_payload(rng, n)
    ref = oracle.ctr_xor(key, iv, pt, threads=THREADS)
    h, ek = oracle.hash_subkey(key), oracle.ek_j0(key, iv)
    ctx = G.gcm_init(key)
    try:
        assert G.gcm_get_ghash_engine(ctx) == G.GCM_GHASH_AUTO
        d_pt, d_aad = dev(pt), dev(aad)
        for m in (n, n - 16):
            d_ct = torch.full((m,), 0xEE, dtype=torch.uint8, device="cuda")
            tag = G.gcm_encrypt(ctx, iv, d_aad, d_pt[:m], d_ct)
            assert np.array_equal(d_ct.cpu().numpy(), ref[:m]), (klen, m, "ciphertext")
            s = oracle.ghash_segmented(h, aad, ref[:m], 1 << 16, THREADS)
            assert bytes(tag) == bytes(x ^ y for x, y in zip(s, ek)), (klen, m, "tag")
            d_back = torch.empty(m, dtype=torch.uint8, device="cuda")
            assert G.gcm_decrypt_verify(ctx, iv, d_aad, d_ct, d_back, tag) == G.GCM_OK
            assert torch.equal(d_back, d_pt[:m])
    finally:
        G.gcm_destroy(ctx)


def test_tc2_chain_random_shapes(G, oracle):
    """40 seeded random shapes through the gcm_tc2 chain (engine TENSOR): lengths 8 .. 24 MiB with any byte count, AAD of
    0 .. 6000 bytes (above 4 KB the head link no longer fits the latency kernel and runs on the row kernel), random grid,
    key size, encrypt or decrypt; every byte and the tag against the oracle."""
    import workloads
    rng = np.random.default_rng(9997)
    for i in range(40):
        klen = 16 if rng.integers(0, 2) else 32
        n = int(rng.integers(8 << 20, 24 << 20))
        a = int(rng.integers(0, 6001)) if i % 4 else 0
        grid = int(rng.choice([0, 0, 1, 17, 148, 400]))
        key, iv, aad = rnd(rng, klen).tobytes(), rnd(rng, 12).tobytes(), rnd(rng, a)
        pt = workloads.random_payload(rng, n)
        want_ct, want_tag = oracle_encrypt(oracle, key, iv, aad, pt)
        ctx = G.gcm_init(key)
        try:
            G.gcm_set_geometry(ctx, grid, 0)
            G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)
            d_aad = dev(aad) if a else None
            if i % 2 == 0:
                d_ct = torch.empty(n, dtype=torch.uint8, device="cuda")
                tag = G.gcm_encrypt(ctx, iv, d_aad, dev(pt), d_ct)
                assert np.array_equal(d_ct.cpu().numpy(), want_ct), (i, klen, n, a, grid, "ciphertext")
                assert bytes(tag) == want_tag, (i, klen, n, a, grid, "tag")
            else:
                d_pt = torch.empty(n, dtype=torch.uint8, device="cuda")
                assert G.gcm_decrypt_verify(ctx, iv, d_aad, dev(want_ct), d_pt, want_tag) == G.GCM_OK, (i, klen, n, a, grid)
                assert np.array_equal(d_pt.cpu().numpy(), pt), (i, klen, n, a, grid, "plaintext")
        finally:
            G.gcm_destroy(ctx)


def test_tensor_kernels_of_several_contexts_on_several_streams(G, oracle):
    """Three contexts (own keys, own scratch and chain slots) on three streams at the same time, all asynchronous: two run
    gcm_tc2 chains (encrypt, then decrypt of what was just written), the third the GHASH-only tensor kernel, three rounds
    without a host synchronisation in between.  Every kernel of these paths takes all 512 TMEM columns of its SM and most
    of its shared memory, so CTAs of different launches queue for SMs; results must not depend on how they interleave."""
    import workloads
    rng = np.random.default_rng(4242)
    n = (9 << 20) + 48
    streams = [torch.cuda.Stream() for _ in range(3)]
    jobs = []
    for j in range(3):
        key = rnd(rng, 32 if j != 1 else 16).tobytes()
        ctx = G.gcm_init(key)
        G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)
        rounds = []
        for r in range(3):
            iv, aad, pt = rnd(rng, 12).tobytes(), rnd(rng, 100 * j + r), workloads.random_payload(rng, n)
            rounds.append({"iv": iv, "aad": aad, "pt": pt, "d_aad": dev(aad) if len(aad) else None, "d_pt": dev(pt),
                           "d_ct": torch.empty(n, dtype=torch.uint8, device="cuda"), "d_back": torch.empty(n, dtype=torch.uint8, device="cuda"),
                           "d_tag": torch.zeros(16, dtype=torch.uint8, device="cuda"), "d_status": torch.full((1,), 9, dtype=torch.int32, device="cuda"),
                           "d_gh": torch.zeros(16, dtype=torch.uint8, device="cuda")})
        jobs.append((key, ctx, rounds))
    torch.cuda.synchronize()
    try:
        for r in range(3):
            for j, (key, ctx, rounds) in enumerate(jobs):
                x = rounds[r]
                if j < 2:
                    G.gcm_encrypt_async(ctx, x["iv"], x["d_aad"], x["d_pt"], x["d_ct"], x["d_tag"], stream=streams[j])
                    G.gcm_decrypt_verify_async(ctx, x["iv"], x["d_aad"], x["d_ct"], x["d_back"], x["d_tag"], x["d_status"], stream=streams[j])
                else:
                    G.gcm_ghash_async(ctx, x["d_aad"], x["d_pt"], x["d_gh"], stream=streams[j])
        torch.cuda.synchronize()
        for j, (key, ctx, rounds) in enumerate(jobs):
            for r, x in enumerate(rounds):
                if j < 2:
                    want_ct, want_tag = oracle_encrypt(oracle, key, x["iv"], x["aad"], x["pt"])
                    assert np.array_equal(x["d_ct"].cpu().numpy(), want_ct), (j, r)
                    assert x["d_tag"].cpu().numpy().tobytes() == want_tag, (j, r)
                    assert int(x["d_status"].item()) == 0 and torch.equal(x["d_back"], x["d_pt"]), (j, r)
                else:
                    h = oracle.hash_subkey(key)
                    assert x["d_gh"].cpu().numpy().tobytes() == bytes(oracle.ghash_segmented(h, x["aad"], x["pt"], 1 << 16, THREADS)), (j, r)
    finally:
        for _, ctx, _ in jobs:
            G.gcm_destroy(ctx)


def test_tc2_kernel_reports_its_own_clock(G):
    """gcm_debug_tc2_clock: refused before the context has run a gcm_tc2 chain; afterwards the SM clock measured by the
    kernel itself (clock64 against %globaltimer over CTA 0's life) is a plausible B200 clock and its duration is
    below the host-timed duration of the whole call."""
    import time
    ctx = G.gcm_init(bytes(range(32)))
    try:
        with pytest.raises(G.GcmError) as e:
            G.gcm_debug_tc2_clock(ctx)
        assert e.value.code == G.GCM_ERR_ARG
        G.gcm_set_ghash_engine(ctx, G.GCM_GHASH_TENSOR)
        n = 64 << 20
        pt = torch.zeros(n, dtype=torch.uint8, device="cuda")
        ct = torch.empty_like(pt)
        G.gcm_encrypt(ctx, bytes(12), None, pt, ct)                     # warm
        t0 = time.perf_counter()
        G.gcm_encrypt(ctx, bytes(12), None, pt, ct)
        wall_ms = (time.perf_counter() - t0) * 1e3
        mhz, ms = G.gcm_debug_tc2_clock(ctx)
        assert 1000.0 < mhz < 2300.0, mhz
        assert 0.0 < ms < wall_ms, (ms, wall_ms)
    finally:
        G.gcm_destroy(ctx)
