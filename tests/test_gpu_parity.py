"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, bit-exact.

Integer / byte work only: the bar is equality of every ciphertext byte and every tag byte.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


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


def check_message(G, oracle, ctx, key, iv, aad, pt, note=""):
    d_aad = dev(aad) if len(aad) else None
    d_pt = dev(pt)
    d_ct = torch.empty_like(d_pt)
    tag = G.gcm_encrypt(ctx, iv, d_aad, d_pt, d_ct)
    ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
    got = d_ct.cpu().numpy()
    assert np.array_equal(got, ref_ct), "ciphertext mismatch %s" % note
    assert tag == ref_tag, "tag mismatch %s" % note
    d_back = torch.empty_like(d_pt)
    rc = G.gcm_decrypt_verify(ctx, iv, d_aad, d_ct, d_back, tag)
    assert rc == G.GCM_OK, note
    assert np.array_equal(d_back.cpu().numpy(), np.asarray(pt)), "roundtrip %s" % note
    return d_aad, d_ct, tag


@pytest.mark.parametrize("klen", [16, 32])
def test_setup_kernel_hash_subkey(G, oracle, klen):
    rng = np.random.default_rng(9000 + klen)
    for _ in range(3):
        key = rnd(rng, klen).tobytes()
        ctx = G.gcm_init(key)
        try:
            assert G.gcm_get_hash_subkey(ctx) == oracle.hash_subkey(key)
        finally:
            G.gcm_destroy(ctx)


@pytest.mark.parametrize("klen", [16, 32])
def test_small_lengths_default_geometry(G, oracle, klen):
    rng = np.random.default_rng(9100 + klen)
    key = rnd(rng, klen).tobytes()
    ctx = G.gcm_init(key)
    try:
        sizes = [(0, 0), (0, 1), (0, 16), (0, 2880), (1, 0), (15, 0), (16, 0), (17, 5), (31, 16), (32, 17),
                 (100, 40), (8191, 0), (8192, 0), (8193, 16), (8192 - 16, 16), (8192 * 3 + 7, 2880),
                 (65536, 256), (100003, 33)]
        for (n, a) in sizes:
            iv = rnd(rng, 12).tobytes()
            check_message(G, oracle, ctx, key, iv, rnd(rng, a), rnd(rng, n), "len=%d aad=%d" % (n, a))
    finally:
        G.gcm_destroy(ctx)


@pytest.mark.parametrize("klen", [16, 32])
def test_geometry_agnostic(G, oracle, klen):
    """the result never depends on the launch geometry.  Small grids force
    long per-thread chains, ragged last rows and every CTA-correction exponent."""
    rng = np.random.default_rng(9200 + klen)
    key = rnd(rng, klen).tobytes()
    iv = rnd(rng, 12).tobytes()
    aad = rnd(rng, 2880)
    pt = rnd(rng, 16 * 512 * 11 + 16 * 77 + 5)
    ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
    ctx = G.gcm_init(key)
    try:
        d_aad, d_pt = dev(aad), dev(pt)
        for (grid, threads) in [(1, 512), (1, 256), (1, 384), (2, 512), (3, 256), (5, 512), (5, 384), (7, 256),
                                (148, 512), (148, 256), (148, 384), (200, 512), (301, 384), (0, 0)]:
            G.gcm_set_geometry(ctx, grid, threads)
            d_ct = torch.empty_like(d_pt)
            tag = G.gcm_encrypt(ctx, iv, d_aad, d_pt, d_ct)
            assert np.array_equal(d_ct.cpu().numpy(), ref_ct), (grid, threads)
            assert tag == ref_tag, (grid, threads)
            d_back = torch.empty_like(d_pt)
            assert G.gcm_decrypt_verify(ctx, iv, d_aad, d_ct, d_back, tag) == G.GCM_OK
            assert np.array_equal(d_back.cpu().numpy(), pt)
    finally:
        G.gcm_destroy(ctx)


def test_many_lengths_small_geometry(G, oracle):
    """Every length 0..700 bytes region and block counts around row boundaries with grid=2, 256
    threads, so rows, pads and tails of every shape occur."""
    rng = np.random.default_rng(9300)
    key = rnd(rng, 16).tobytes()
    ctx = G.gcm_init(key)
    try:
        G.gcm_set_geometry(ctx, 2, 256)
        lens = list(range(0, 70)) + [16 * 255, 16 * 256 - 1, 16 * 256, 16 * 256 + 1, 16 * 257, 16 * 511 + 3,
                                       16 * 512, 16 * 513 - 15, 16 * 1024, 16 * 1025 + 9, 16 * 2047, 16 * 2049]
        for n in lens:
            for a in (0, 7, 16, 100):
                iv = rnd(rng, 12).tobytes()
                check_message(G, oracle, ctx, key, iv, rnd(rng, a), rnd(rng, n), "len=%d aad=%d" % (n, a))
    finally:
        G.gcm_destroy(ctx)


@pytest.mark.parametrize("klen", [16, 32])
def test_latency_kernel_every_shape(G, oracle, klen):
    """Messages of at most 511 GHASH blocks take the single-CTA latency kernel (gcm_small.cu) under the default
    geometry: every payload length 0..130, AAD lengths around block edges, the boundary to the fused kernel
    (510, 511, 512 blocks), unaligned and in-place buffers with guard regions, and every tamper kind."""
    rng = np.random.default_rng(9350 + klen)
    key = rnd(rng, klen).tobytes()
    ctx = G.gcm_init(key)
    try:
        for n in range(0, 131):
            a = (0, 1, 15, 16, 17, 33, 256)[n % 7]
            check_message(G, oracle, ctx, key, rnd(rng, 12).tobytes(), rnd(rng, a), rnd(rng, n), "len=%d aad=%d" % (n, a))
        for blocks, a in [(508, 16), (509, 16), (510, 16), (509, 0), (510, 0), (511, 0), (329, 2880), (330, 2880), (331, 2871)]:
            for tail in (0, 5):
                n = 16 * blocks - tail
                check_message(G, oracle, ctx, key, rnd(rng, 12).tobytes(), rnd(rng, a), rnd(rng, n), "blocks=%d aad=%d" % (blocks, a))
        # unaligned input / output / AAD, nothing written outside the output range
        iv, aad, n = rnd(rng, 12).tobytes(), rnd(rng, 45), 16 * 200 + 9
        pt = rnd(rng, n)
        ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
        for (oi, oo, oa) in [(0, 0, 0), (1, 0, 0), (0, 3, 0), (5, 5, 1), (15, 9, 7)]:
            big_in = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
            big_out = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
            big_aad = torch.zeros(len(aad) + 16, dtype=torch.uint8, device="cuda")
            big_in[oi: oi + n] = dev(pt)
            big_aad[oa: oa + len(aad)] = dev(aad)
            tag = G.gcm_encrypt(ctx, iv, big_aad[oa: oa + len(aad)], big_in[oi: oi + n], big_out[oo: oo + n])
            out = big_out.cpu().numpy()
            assert tag == ref_tag and np.array_equal(out[oo: oo + n], ref_ct), (oi, oo, oa)
            assert not out[:oo].any() and not out[oo + n:].any(), "wrote outside the output range"
        buf = dev(pt).clone()
        assert G.gcm_encrypt(ctx, iv, dev(aad), buf, buf) == ref_tag and np.array_equal(buf.cpu().numpy(), ref_ct)   # in place
        assert G.gcm_decrypt_verify(ctx, iv, dev(aad), buf, buf, ref_tag) == G.GCM_OK
        assert np.array_equal(buf.cpu().numpy(), pt)
        # tamper: ciphertext, tag, AAD, IV, length -> GCM_ERR_AUTH and an all-zero output
        d_aad, d_ct = dev(aad), dev(ref_ct)

        def rejected(iv_=iv, aad_=d_aad, ct_=d_ct, tag_=ref_tag):
            out = torch.full((ct_.numel(),), 0xAA, dtype=torch.uint8, device="cuda")
            return G.gcm_decrypt_verify(ctx, iv_, aad_, ct_, out, tag_) == G.GCM_ERR_AUTH and not bool(out.any().item())

        for pos in (0, n // 2, n - 1):
            bad = d_ct.clone(); bad[pos] ^= 0x10
            assert rejected(ct_=bad)
        t = bytearray(ref_tag); t[15] ^= 0x80
        assert rejected(tag_=bytes(t))
        bad_aad = d_aad.clone(); bad_aad[44] ^= 1
        assert rejected(aad_=bad_aad) and rejected(aad_=d_aad[:-1].clone()) and rejected(ct_=d_ct[:-1].clone())
        v = bytearray(iv); v[0] ^= 2
        assert rejected(iv_=bytes(v))
        # async form on the latency kernel: device tag in, status word out, gated wipe
        d_tag = dev(np.frombuffer(ref_tag, np.uint8))
        d_status = torch.full((1,), -7, dtype=torch.int32, device="cuda")
        out = torch.full((n,), 0x55, dtype=torch.uint8, device="cuda")
        bad = d_ct.clone(); bad[3] ^= 1
        G.gcm_decrypt_verify_async(ctx, iv, d_aad, bad, out, d_tag, d_status)
        torch.cuda.synchronize()
        assert int(d_status.item()) == G.GCM_ERR_AUTH and not bool(out.any().item())
        G.gcm_decrypt_verify_async(ctx, iv, d_aad, d_ct, out, d_tag, d_status)
        torch.cuda.synchronize()
        assert int(d_status.item()) == G.GCM_OK and np.array_equal(out.cpu().numpy(), pt)
        # the same messages through the fused kernel (explicit geometry) give the same bytes
        G.gcm_set_geometry(ctx, 3, 256)
        d_out = torch.empty(n, dtype=torch.uint8, device="cuda")
        assert G.gcm_encrypt(ctx, iv, d_aad, dev(pt), d_out) == ref_tag and np.array_equal(d_out.cpu().numpy(), ref_ct)
    finally:
        G.gcm_destroy(ctx)


def test_in_place_and_unaligned(G, oracle):
    rng = np.random.default_rng(9400)
    key = rnd(rng, 32).tobytes()
    iv = rnd(rng, 12).tobytes()
    aad = rnd(rng, 50)
    n = 16 * 512 * 3 + 100
    pt = rnd(rng, n)
    ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
    ctx = G.gcm_init(key)
    try:
        d_aad = dev(aad)
        buf = dev(pt).clone()
        tag = G.gcm_encrypt(ctx, iv, d_aad, buf, buf)          # in place
        assert tag == ref_tag and np.array_equal(buf.cpu().numpy(), ref_ct)
        assert G.gcm_decrypt_verify(ctx, iv, d_aad, buf, buf, tag) == G.GCM_OK
        assert np.array_equal(buf.cpu().numpy(), pt)
        for (oi, oo, oa) in [(1, 0, 0), (0, 3, 0), (5, 5, 1), (15, 9, 7)]:
            big_in = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
            big_out = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
            big_aad = torch.zeros(len(aad) + 16, dtype=torch.uint8, device="cuda")
            big_in[oi: oi + n] = dev(pt)
            big_aad[oa: oa + len(aad)] = d_aad
            tag = G.gcm_encrypt(ctx, iv, big_aad[oa: oa + len(aad)], big_in[oi: oi + n], big_out[oo: oo + n])
            out = big_out.cpu().numpy()
            assert tag == ref_tag, (oi, oo, oa)
            assert np.array_equal(out[oo: oo + n], ref_ct), (oi, oo, oa)
            assert not out[:oo].any() and not out[oo + n:].any(), "wrote outside the output range"
        # partial overlap is refused
        big = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
        with pytest.raises(G.GcmError) as e:
            G.gcm_encrypt(ctx, iv, d_aad, big[0:n], big[16: 16 + n])
        assert e.value.code == G.GCM_ERR_ARG
    finally:
        G.gcm_destroy(ctx)


@pytest.mark.parametrize("klen", [16, 32])
def test_tamper_detection_and_suppression(G, oracle, klen):
    """PAPER.md L219 (validation gate), L243 (payload zero-filled), L157 (AAD binding)."""
    rng = np.random.default_rng(9500 + klen)
    key = rnd(rng, klen).tobytes()
    iv = rnd(rng, 12).tobytes()
    aad = rnd(rng, 2880)
    pt = rnd(rng, 16 * 512 * 2 + 33)
    ctx = G.gcm_init(key)
    try:
        d_aad, d_ct, tag = check_message(G, oracle, ctx, key, iv, aad, pt)
        n = len(pt)

        def rejected(iv_=iv, aad_=d_aad, ct_=d_ct, tag_=tag):
            out = torch.full((ct_.numel(),), 0xAA, dtype=torch.uint8, device="cuda")
            rc = G.gcm_decrypt_verify(ctx, iv_, aad_, ct_, out, tag_)
            return rc == G.GCM_ERR_AUTH and not bool(out.any().item())

        for pos in (0, n // 2, n - 1):
            bad = d_ct.clone(); bad[pos] ^= 0x04
            assert rejected(ct_=bad)
        for bit in (0, 63, 127):
            t = bytearray(tag); t[bit // 8] ^= 1 << (bit % 8)
            assert rejected(tag_=bytes(t))
        bad_aad = d_aad.clone(); bad_aad[100] ^= 1
        assert rejected(aad_=bad_aad)
        assert rejected(aad_=d_aad[:-1].clone())
        v = bytearray(iv); v[11] ^= 1
        assert rejected(iv_=bytes(v))
        assert rejected(ct_=d_ct[:-1].clone())
        # the oracle agrees on rejection and on zeros
        bad = d_ct.clone(); bad[7] ^= 0x80
        ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)     # the oracle's own ciphertext, same flip
        ref_bad = ref_ct.copy(); ref_bad[7] ^= 0x80
        rc, out = oracle.gcm_decrypt_verify(key, iv, aad, ref_bad, ref_tag)
        assert rc == oracle.AUTH_FAIL and not out.any()
        # async form: status word + wipe kernel on the stream
        d_tag = dev(np.frombuffer(tag, np.uint8))
        d_status = torch.full((1,), -7, dtype=torch.int32, device="cuda")
        out = torch.full((n,), 0x55, dtype=torch.uint8, device="cuda")
        G.gcm_decrypt_verify_async(ctx, iv, d_aad, bad, out, d_tag, d_status)
        torch.cuda.synchronize()
        assert int(d_status.item()) == G.GCM_ERR_AUTH and not bool(out.any().item())
        G.gcm_decrypt_verify_async(ctx, iv, d_aad, d_ct, out, d_tag, d_status)
        torch.cuda.synchronize()
        assert int(d_status.item()) == G.GCM_OK and np.array_equal(out.cpu().numpy(), pt)
    finally:
        G.gcm_destroy(ctx)


def test_async_encrypt_and_ghash_only(G, oracle):
    rng = np.random.default_rng(9600)
    key = rnd(rng, 32).tobytes()
    iv = rnd(rng, 12).tobytes()
    aad = rnd(rng, 77)
    pt = rnd(rng, 16 * 512 * 5 + 9)
    ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
    ctx = G.gcm_init(key)
    try:
        d_aad, d_pt = dev(aad), dev(pt)
        d_ct = torch.empty_like(d_pt)
        d_tag = torch.zeros(16, dtype=torch.uint8, device="cuda")
        G.gcm_encrypt_async(ctx, iv, d_aad, d_pt, d_ct, d_tag)
        torch.cuda.synchronize()
        assert np.array_equal(d_ct.cpu().numpy(), ref_ct)
        assert d_tag.cpu().numpy().tobytes() == ref_tag
        d_s = torch.zeros(16, dtype=torch.uint8, device="cuda")
        G.gcm_ghash_async(ctx, d_aad, d_ct, d_s)
        torch.cuda.synchronize()
        assert d_s.cpu().numpy().tobytes() == oracle.ghash(oracle.hash_subkey(key), aad, ref_ct)
    finally:
        G.gcm_destroy(ctx)


def test_error_codes(G):
    ctx = G.gcm_init(bytes(16))
    try:
        t = torch.zeros(32, dtype=torch.uint8, device="cuda")
        import ctypes
        from paper_2602_23067_b200 import gcm as B
        tag = ctypes.create_string_buffer(16)
        # length limit
        assert B._L.gcm_encrypt(ctx, bytes(12), None, 0, t.data_ptr(), (1 << 36) - 31, t.data_ptr(), tag, None) == G.GCM_ERR_LEN
        # NULL data with non-zero length
        assert B._L.gcm_encrypt(ctx, bytes(12), None, 5, t.data_ptr(), 16, t.data_ptr(), tag, None) == G.GCM_ERR_ARG
        assert B._L.gcm_encrypt(ctx, None, None, 0, t.data_ptr(), 16, t.data_ptr(), tag, None) == G.GCM_ERR_ARG
        with pytest.raises(G.GcmError):
            G.gcm_set_geometry(ctx, 5, 100)
    finally:
        G.gcm_destroy(ctx)


def test_config_c1_full(G, oracle):
    m = workloads.config_c1()
    ctx = G.gcm_init(m.key)
    try:
        check_message(G, oracle, ctx, m.key, m.iv, m.aad, m.payload, "C1")
    finally:
        G.gcm_destroy(ctx)


def test_config_c3_scaled_batch(G, oracle):
    msgs = workloads.config_c3(n_images=4, ny=512, nx=384, n_sources=20)
    batch = []
    for m in msgs:
        d_in = dev(m.payload)
        batch.append({"key": m.key, "iv": m.iv, "aad": dev(m.aad), "input": d_in, "output": torch.empty_like(d_in)})
    tags = G.gcm_encrypt_batch(batch)
    for m, b, tag in zip(msgs, batch, tags):
        ref_ct, ref_tag = oracle.gcm_encrypt(m.key, m.iv, m.aad, m.payload)
        assert tag == ref_tag, m.name
        assert np.array_equal(b["output"].cpu().numpy(), ref_ct), m.name
    # structured plaintext must still look like noise: no repeated ciphertext block
    ct0 = batch[0]["output"].cpu().numpy()
    blocks = ct0[: ct0.size // 16 * 16].reshape(-1, 16)
    assert len({bytes(b) for b in blocks[:20000]}) == min(20000, len(blocks))
    dec = []
    for b, tag in zip(batch, tags):
        dec.append({"key": b["key"], "iv": b["iv"], "aad": b["aad"], "input": b["output"],
                    "output": torch.empty_like(b["output"]), "tag": tag})
    dec[2]["tag"] = bytes(16)
    st = G.gcm_decrypt_verify_batch(dec)
    assert st == [G.GCM_OK, G.GCM_OK, G.GCM_ERR_AUTH, G.GCM_OK]
    for i, (m, d) in enumerate(zip(msgs, dec)):
        got = d["output"].cpu().numpy()
        if i == 2:
            assert not got.any()
        else:
            assert np.array_equal(got, m.payload)
    G.gcm_batch_release()


def test_config_c4_scaled_batch(G, oracle):
    msgs = workloads.config_c4(n_messages=60, max_len=20000)
    batch = []
    for m in msgs:
        d_in = dev(m.payload)
        batch.append({"key": m.key, "iv": m.iv, "aad": dev(m.aad) if m.aad.size else None,
                      "input": d_in, "output": torch.empty_like(d_in)})
    tags = G.gcm_encrypt_batch(batch)
    for m, b, tag in zip(msgs, batch, tags):
        ref_ct, ref_tag = oracle.gcm_encrypt(m.key, m.iv, m.aad, m.payload)
        assert tag == ref_tag, m.name
        assert np.array_equal(b["output"].cpu().numpy(), ref_ct), m.name
    G.gcm_batch_release()


def test_batch_warp_per_message_kernel(G, oracle):
    """The one-warp-per-message kernel: both key sizes in one call, every tail shape, empty messages,
    empty AAD, unaligned buffers, messages packed in one buffer at 16-byte offsets (config C4's layout),
    then decrypt_verify with a few tampered messages: rejected, zero-filled, neighbours untouched."""
    rng = np.random.default_rng(9650)
    lens = [0, 1, 15, 16, 17, 31, 32, 33, 495, 496, 497, 511, 512, 513, 1023, 1024, 4096, 8191, 8192 + 5,
            16 * 32 * 7, 16 * 32 * 7 + 16 * 30, 16 * 32 * 7 + 16 * 30 + 9, 65536, 70001, 200000]
    lens += rng.integers(1, 65537, 40).tolist()
    specs = []
    for i, n in enumerate(lens):
        klen = 16 if i % 3 else 32
        a = [0, 1, 16, 17, 100, 256, 2880][i % 7]
        specs.append((rnd(rng, klen).tobytes(), rnd(rng, 12).tobytes(), rnd(rng, a), rnd(rng, n), i % 5 == 4))
    # one packed buffer; unaligned messages start 3 bytes past a 16-byte boundary
    offs, pos = [], 0
    for (_, _, _, pt, unal) in specs:
        pos = (pos + 15) // 16 * 16 + (3 if unal else 0)
        offs.append(pos)
        pos += len(pt) + 16            # a guard gap after every message
    big_in = torch.zeros(pos + 16, dtype=torch.uint8, device="cuda")
    big_out = torch.zeros(pos + 16, dtype=torch.uint8, device="cuda")
    for (_, _, _, pt, _), o in zip(specs, offs):
        if len(pt):
            big_in[o: o + len(pt)] = dev(pt)
    batch = []
    for (key, iv, aad, pt, _), o in zip(specs, offs):
        batch.append({"key": key, "iv": iv, "aad": dev(aad) if len(aad) else None,
                      "input": big_in[o: o + len(pt)], "output": big_out[o: o + len(pt)]})
    tags = G.gcm_encrypt_batch(batch)
    out = big_out.cpu().numpy()
    covered = np.zeros(out.size, bool)
    for (key, iv, aad, pt, _), o, tag in zip(specs, offs, tags):
        ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
        assert tag == ref_tag, "tag len=%d aad=%d" % (len(pt), len(aad))
        assert np.array_equal(out[o: o + len(pt)], ref_ct), "ct len=%d aad=%d" % (len(pt), len(aad))
        covered[o: o + len(pt)] = True
    assert not out[~covered].any(), "wrote outside a message's output range"
    # decrypt: tamper message 5 (tag), 9 (ciphertext), 20 (aad), 24 (last byte of a 200000-byte message)
    dec_out = torch.full_like(big_out, 0x77)
    dec = []
    for i, (b, tag) in enumerate(zip(batch, tags)):
        o, n = offs[i], len(specs[i][3])
        dec.append({"key": b["key"], "iv": b["iv"], "aad": b["aad"], "input": big_out[o: o + n],
                    "output": dec_out[o: o + n], "tag": tag})
    bad = {5, 9, 20, 24}
    t = bytearray(tags[5]); t[15] ^= 1; dec[5]["tag"] = bytes(t)
    big_out[offs[9] + len(specs[9][3]) // 2] ^= 0x10
    a20 = dec[20]["aad"].clone(); a20[0] ^= 0x80; dec[20]["aad"] = a20
    big_out[offs[24] + len(specs[24][3]) - 1] ^= 1
    st = G.gcm_decrypt_verify_batch(dec)
    got = dec_out.cpu().numpy()
    for i, (spec, o) in enumerate(zip(specs, offs)):
        n = len(spec[3])
        if i in bad:
            assert st[i] == G.GCM_ERR_AUTH, i
            assert not got[o: o + n].any(), "message %d not suppressed" % i
        else:
            assert st[i] == G.GCM_OK, i
            assert np.array_equal(got[o: o + n], spec[3]), i
    assert (got[~covered] == 0x77).all()
    # argument errors are reported per message and do not stop the others
    batch2 = [dict(batch[1]), dict(batch[2])]
    batch2[0]["key"] = bytes(24)
    with pytest.raises(G.GcmError) as e:
        G.gcm_encrypt_batch(batch2)
    assert e.value.code == G.GCM_ERR_ARG
    G.gcm_batch_release()


def test_host_buffers_single_chunk(G, oracle):
    rng = np.random.default_rng(9700)
    key = rnd(rng, 32).tobytes()
    ctx = G.gcm_init(key)
    try:
        for (n, a) in [(0, 0), (0, 40), (1, 0), (100003, 2880), (16 * 512 * 4, 16)]:
            iv = rnd(rng, 12).tobytes()
            aad, pt = rnd(rng, a), rnd(rng, n)
            h_pt = torch.from_numpy(pt.copy()).pin_memory()
            h_ct = torch.empty(n, dtype=torch.uint8).pin_memory()
            tag = G.gcm_encrypt_host(ctx, iv, aad, h_pt, h_ct)
            ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
            assert tag == ref_tag and np.array_equal(h_ct.numpy(), ref_ct), (n, a)
            back = np.empty(n, np.uint8)                       # pageable output also works
            assert G.gcm_decrypt_verify_host(ctx, iv, aad, h_ct, back, tag) == G.GCM_OK
            assert np.array_equal(back, pt)
            if n:
                bad = h_ct.clone(); bad[n // 2] ^= 1
                assert G.gcm_decrypt_verify_host(ctx, iv, aad, bad, back, tag) == G.GCM_ERR_AUTH
                assert not back.any()
    finally:
        G.gcm_destroy(ctx)


def test_host_pipeline_multi_chunk(G, oracle):
    """192 MiB + 12345 bytes through the chunk pipeline (about eight chunks, the last one ragged): the running
    GHASH state is chained across chunks and the counters continue across chunk boundaries."""
    import os
    rng = np.random.default_rng(9800)
    key = rnd(rng, 32).tobytes()
    iv = rnd(rng, 12).tobytes()
    aad = rnd(rng, 2880)
    n = 3 * (64 << 20) + 12345
    pt = workloads.random_payload(rng, n)
    ctx = G.gcm_init(key)
    try:
        h_pt = torch.from_numpy(pt.copy()).pin_memory()
        h_ct = torch.empty(n, dtype=torch.uint8).pin_memory()
        tag = G.gcm_encrypt_host(ctx, iv, aad, h_pt, h_ct)
        # same bytes through the single-launch device path
        d_ct = torch.empty(n, dtype=torch.uint8, device="cuda")
        tag_dev = G.gcm_encrypt(ctx, iv, dev(aad), h_pt.cuda(), d_ct)
        assert tag == tag_dev and torch.equal(d_ct.cpu(), h_ct)
        # and against the oracle (CTR over the host cores, GHASH by the pinned segment identity)
        ref_ct, ref_tag = oracle.gcm_encrypt_threaded(key, iv, aad, pt, threads=os.cpu_count() or 1, segment_blocks=1 << 16)
        assert tag == ref_tag
        assert np.array_equal(h_ct.numpy(), ref_ct)
        back = torch.empty(n, dtype=torch.uint8).pin_memory()
        assert G.gcm_decrypt_verify_host(ctx, iv, aad, h_ct, back, tag) == G.GCM_OK
        assert torch.equal(back, h_pt)
        h_ct[(64 << 20) + 5] ^= 0x20
        assert G.gcm_decrypt_verify_host(ctx, iv, aad, h_ct, back, tag) == G.GCM_ERR_AUTH
        assert not bool(back.any().item())
    finally:
        G.gcm_destroy(ctx)


def test_pipe_rate_probe(G):
    """gcm_measure_pipe_rates: the shared-memory data pipe serves one 128-byte wavefront per SM-cycle
    (32 four-byte or 8 sixteen-byte lookups), the ALU and FMA pipes 64 lanes each."""
    r = G.gcm_measure_pipe_rates()
    assert set(r) == set(G.RATE_NAMES)
    assert 24 <= r["lds32"] <= 33 and 6 <= r["lds128"] <= 8.3
    assert 48 <= r["lop3"] <= 66 and 48 <= r["prmt"] <= 66 and 48 <= r["imad"] <= 66
    assert r["lop3_imad"] > r["lop3"]


def test_host_pipeline_chunk_plan_boundaries(G, oracle):
    """The host pipeline cuts a message into chunks of 2 MiB at both ends, doubling towards the middle; the GHASH
    state, the chunk powers and the counters have to line up at every cut.  Sizes on and around the cuts (one, two,
    three ... chunks, a ragged last chunk of 1 byte, of 2 MiB - 1), with and without AAD, encrypt and decrypt."""
    import os
    rng = np.random.default_rng(9850)
    key = rnd(rng, 16).tobytes()
    MiB = 1 << 20
    sizes = [2 * MiB - 1, 2 * MiB, 2 * MiB + 1, 4 * MiB, 4 * MiB + 17, 6 * MiB - 1, 6 * MiB + 16, 10 * MiB + 5,
             14 * MiB, 24 * MiB + 1, 26 * MiB - 16, 40 * MiB + 123457]
    ctx = G.gcm_init(key)
    try:
        for i, n in enumerate(sizes):
            iv = rnd(rng, 12).tobytes()
            aad = rnd(rng, [0, 16, 2880, 45][i % 4])
            pt = workloads.random_payload(rng, n)
            ref_ct, ref_tag = oracle.gcm_encrypt_threaded(key, iv, aad, pt, threads=os.cpu_count() or 1, segment_blocks=1 << 14)
            h_pt = torch.from_numpy(pt.copy()).pin_memory()
            h_ct = torch.empty(n, dtype=torch.uint8).pin_memory()
            tag = G.gcm_encrypt_host(ctx, iv, aad, h_pt, h_ct)
            assert tag == ref_tag, n
            assert np.array_equal(h_ct.numpy(), ref_ct), n
            back = torch.empty(n, dtype=torch.uint8).pin_memory()
            assert G.gcm_decrypt_verify_host(ctx, iv, aad, h_ct, back, tag) == G.GCM_OK, n
            assert torch.equal(back, h_pt), n
            assert G.gcm_decrypt_verify_host_strict(ctx, iv, aad, h_ct, back, tag) == G.GCM_OK, n
            h_ct[n - 1] ^= 1
            assert G.gcm_decrypt_verify_host(ctx, iv, aad, h_ct, back, tag) == G.GCM_ERR_AUTH, n
            assert not bool(back.any().item())
    finally:
        G.gcm_destroy(ctx)


def test_random_shapes_against_the_oracle(G, oracle):
    """Differential run over 240 seeded random shapes: length (skewed towards row and block edges), AAD length,
    key size, source / destination / AAD misalignment, in place or not, launch geometry (threads 256 / 384 / 512, 1-300
    CTAs, or the default with its latency-kernel switch), encrypt then decrypt_verify, every byte and tag against the
    oracle, nothing written outside the output range."""
    rng = np.random.default_rng(9990)
    ctxs = {}
    try:
        for case in range(240):
            klen = 16 if rng.integers(0, 2) else 32
            key = ctxs.get(klen)
            if key is None:
                k = rnd(rng, klen).tobytes()
                ctxs[klen] = key = (k, G.gcm_init(k))
            k, ctx = key
            kind = int(rng.integers(0, 4))
            if kind == 0:
                n = int(rng.integers(0, 600))
            elif kind == 1:
                n = 512 * int(rng.integers(1, 40)) + int(rng.integers(-17, 18))
            elif kind == 2:
                n = 16 * int(rng.integers(1, 20000)) + int(rng.integers(0, 16))
            else:
                n = int(rng.integers(1, 1 << 20))
            n = max(n, 0)
            a = int(rng.choice([0, 0, 1, 15, 16, 17, 45, 256, 2880, int(rng.integers(0, 4000))]))
            oi, oo, oa = (int(rng.integers(0, 16)) if rng.integers(0, 3) == 0 else 0 for _ in range(3))
            in_place = bool(rng.integers(0, 4) == 0)
            geom = [(0, 0), (0, 0), (1, 256), (3, 384), (7, 512), (148, 384), (int(rng.integers(1, 300)), int(rng.choice([256, 384, 512])))][int(rng.integers(0, 7))]
            G.gcm_set_geometry(ctx, *geom)
            iv, aad, pt = rnd(rng, 12).tobytes(), rnd(rng, a), rnd(rng, n)
            ref_ct, ref_tag = oracle.gcm_encrypt(k, iv, aad, pt)
            big_in = torch.zeros(n + 48, dtype=torch.uint8, device="cuda")
            big_in[oi: oi + n] = dev(pt)
            big_aad = torch.zeros(a + 32, dtype=torch.uint8, device="cuda")
            big_aad[oa: oa + a] = dev(aad)
            if in_place:
                big_out, oo = big_in, oi
            else:
                big_out = torch.zeros(n + 48, dtype=torch.uint8, device="cuda")
            d_aad = big_aad[oa: oa + a] if a else None
            tag = G.gcm_encrypt(ctx, iv, d_aad, big_in[oi: oi + n], big_out[oo: oo + n])
            out = big_out.cpu().numpy()
            note = (case, klen, n, a, oi, oo, oa, in_place, geom)
            assert tag == ref_tag, note
            assert np.array_equal(out[oo: oo + n], ref_ct), note
            assert not out[:oo].any() and not out[oo + n:].any(), note
            back = torch.full((n + 32,), 0x5C, dtype=torch.uint8, device="cuda")
            assert G.gcm_decrypt_verify(ctx, iv, d_aad, big_out[oo: oo + n], back[16: 16 + n], tag) == G.GCM_OK, note
            got = back.cpu().numpy()
            assert np.array_equal(got[16: 16 + n], pt) and (got[:16] == 0x5C).all() and (got[16 + n:] == 0x5C).all(), note
    finally:
        for _, ctx in ctxs.values():
            G.gcm_destroy(ctx)
