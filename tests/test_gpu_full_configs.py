"""GPU parity at BASELINE.json's FULL sizes (configs C2-C5), in the launch configuration bench.py times
(default geometry: one 512-thread CTA per SM), through the C ABI binding, against the CPU oracle.

The oracle is the plain definition; at these sizes it is spread over the host cores only across
*independent* pieces: CTR byte ranges (the counter depends on the block index
only) and GHASH segments combined by the identity pinned against the Horner chain in
tests/test_oracle_ghash.py.  Messages are walked in 128 MiB windows so that host memory stays small.
Bar: every ciphertext byte and every tag byte equal (integer work, bit-exact).
"""
import os

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

THREADS = os.cpu_count() or 1
WINDOW = 128 << 20
SEG_BLOCKS = 1 << 16          # 1 MiB GHASH segments


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2602_23067_b200 as pkg
    return pkg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle_check_device_message(oracle, key, iv, aad, d_pt, d_ct, tag, note):
    """Ciphertext (every byte) and tag of a device-resident message against the oracle, window by
    window: C = P xor E_K(IV || BE32(g + 2)); S = GHASH(A, C) by weighted segments; T = E_K(J0) xor S."""
    n = d_pt.numel()
    n_c = (n + 15) // 16
    n_a = (len(aad) + 15) // 16
    h = oracle.hash_subkey(key)
    acc = np.zeros(16, np.uint8)
    if len(aad):
        acc ^= np.frombuffer(oracle.ghash_segment(h, aad, n_c + 1), np.uint8)
    from concurrent.futures import ThreadPoolExecutor
    for off in range(0, n, WINDOW):
        hi = min(n, off + WINDOW)
        pt = d_pt[off:hi].cpu().numpy()
        ct = d_ct[off:hi].cpu().numpy()
        ref = oracle.ctr_xor(key, iv, pt, first_block=off // 16, threads=THREADS)
        assert np.array_equal(ref, ct), "%s: ciphertext differs in window at byte %d" % (note, off)
        jobs = []
        for s in range(0, hi - off, 16 * SEG_BLOCKS):
            piece = ref[s: s + 16 * SEG_BLOCKS]
            done = (off + s) // 16 + (piece.size + 15) // 16
            jobs.append((piece, n_c - done + 1))
        with ThreadPoolExecutor(THREADS) as ex:
            for part in ex.map(lambda j: oracle.ghash_segment(h, j[0], j[1]), jobs):
                acc ^= np.frombuffer(part, np.uint8)
    lenblk = (8 * len(aad)).to_bytes(8, "big") + (8 * n).to_bytes(8, "big")
    acc ^= np.frombuffer(oracle.ghash_segment(h, lenblk, 0), np.uint8)
    ref_tag = bytes(x ^ y for x, y in zip(acc.tobytes(), oracle.ek_j0(key, iv)))
    assert tag == ref_tag, "%s: tag differs" % note
    assert n_a >= 0


def test_config_c2_full(G, oracle):
    """C2: AES-256-GCM, one 256 MiB uniform message, 2880-byte FITS header block as AAD."""
    m = workloads.config_c2()
    assert m.payload.size == 256 << 20 and m.aad.size == 2880 and len(m.key) == 32
    ctx = G.gcm_init(m.key)
    try:
        d_aad, d_pt = dev(m.aad), dev(m.payload)
        d_ct = torch.empty_like(d_pt)
        tag = G.gcm_encrypt(ctx, m.iv, d_aad, d_pt, d_ct)
        oracle_check_device_message(oracle, m.key, m.iv, m.aad, d_pt, d_ct, tag, "C2")
        d_back = torch.empty_like(d_pt)
        assert G.gcm_decrypt_verify(ctx, m.iv, d_aad, d_ct, d_back, tag) == G.GCM_OK
        assert torch.equal(d_back, d_pt)
    finally:
        G.gcm_destroy(ctx)


def test_config_c3_full_batch(G, oracle):
    """C3: 16 FITS-shaped images of 4096 x 4096 float32 (64 MiB + pad to a 2880-byte multiple), one
    AES-256 key, 16 IVs, per-image header as AAD, batched API."""
    msgs = workloads.config_c3()
    assert len(msgs) == 16 and all(m.payload.size == 67109760 and m.aad.size == 2880 for m in msgs)
    batch = []
    for m in msgs:
        d_in = dev(m.payload)
        batch.append({"key": m.key, "iv": m.iv, "aad": dev(m.aad), "input": d_in, "output": torch.empty_like(d_in)})
    tags = G.gcm_encrypt_batch(batch)
    for m, b, tag in zip(msgs, batch, tags):
        oracle_check_device_message(oracle, m.key, m.iv, m.aad, b["input"], b["output"], tag, m.name)
    # the constant-valued blank regions must not show through: no repeated block
    ct0 = batch[0]["output"][: 16 * 200000].cpu().numpy().reshape(-1, 16)
    assert len({bytes(b) for b in ct0}) == len(ct0)
    dec = [{"key": b["key"], "iv": b["iv"], "aad": b["aad"], "input": b["output"],
            "output": torch.empty_like(b["output"]), "tag": tag} for b, tag in zip(batch, tags)]
    bad = 11
    dec[bad]["input"] = dec[bad]["input"].clone()
    dec[bad]["input"][12345678] ^= 0x10
    st = G.gcm_decrypt_verify_batch(dec)
    assert st == [G.GCM_ERR_AUTH if i == bad else G.GCM_OK for i in range(16)]
    for i, (b, d) in enumerate(zip(batch, dec)):
        if i == bad:
            assert not bool(d["output"].any().item())
        else:
            assert torch.equal(d["output"], b["input"])
    G.gcm_batch_release()


def test_config_c4_full_batch(G, oracle):
    """C4: 10,000 AES-128 messages, len ~ U{1..65536}, AAD len ~ U{0..256}, own key and IV each,
    payloads packed in one device buffer at 16-byte-aligned offsets, batched API."""
    msgs = workloads.config_c4()
    assert len(msgs) == 10000
    offs, total = [], 0
    for m in msgs:
        offs.append(total)
        total += (m.payload.size + 15) // 16 * 16
    aoffs, atotal = [], 0
    for m in msgs:
        aoffs.append(atotal)
        atotal += (m.aad.size + 15) // 16 * 16
    h_in = np.zeros(total, np.uint8)
    h_aad = np.zeros(max(atotal, 16), np.uint8)
    for m, o, ao in zip(msgs, offs, aoffs):
        h_in[o: o + m.payload.size] = m.payload
        h_aad[ao: ao + m.aad.size] = m.aad
    d_in, d_aad = dev(h_in), dev(h_aad)
    d_out = torch.zeros_like(d_in)
    batch = [{"key": m.key, "iv": m.iv, "aad": d_aad[ao: ao + m.aad.size] if m.aad.size else None,
              "input": d_in[o: o + m.payload.size], "output": d_out[o: o + m.payload.size]}
             for m, o, ao in zip(msgs, offs, aoffs)]
    tags = G.gcm_encrypt_batch(batch)
    out = d_out.cpu().numpy()
    from concurrent.futures import ThreadPoolExecutor

    def ref(m):
        return oracle.gcm_encrypt(m.key, m.iv, m.aad, m.payload)

    with ThreadPoolExecutor(THREADS) as ex:
        refs = list(ex.map(ref, msgs))
    for m, o, tag, (ref_ct, ref_tag) in zip(msgs, offs, tags, refs):
        assert tag == ref_tag, m.name
        assert np.array_equal(out[o: o + m.payload.size], ref_ct), m.name
        pad_end = (m.payload.size + 15) // 16 * 16
        assert not out[o + m.payload.size: o + pad_end].any(), "%s: wrote past len" % m.name
    # the same 10,000 messages through the device-descriptor call (ordering on the device, tags in the descriptors)
    d_out2 = torch.zeros_like(d_in)
    host = G.gcm_pack_dmsgs([dict(b, output=d_out2[o: o + m.payload.size]) for b, m, o in zip(batch, msgs, offs)])
    d_msgs = torch.from_numpy(host.view(np.uint8).copy()).cuda()
    G.gcm_encrypt_batch_device(d_msgs)
    torch.cuda.synchronize()
    res = d_msgs.cpu().numpy().view(host.dtype)
    assert torch.equal(d_out2, d_out), "device-descriptor ciphertext differs from the host-descriptor call's"
    assert not res["status"].any()
    for m, (_, ref_tag), i in zip(msgs, refs, range(len(msgs))):
        assert res["tag"][i].tobytes() == ref_tag, m.name
    # decrypt + verify the whole batch, three seeded forgeries (ciphertext, tag, AAD)
    d_back = torch.zeros_like(d_in)
    dec = [{"key": b["key"], "iv": b["iv"], "aad": b["aad"], "input": b["output"],
            "output": d_back[o: o + m.payload.size], "tag": tag}
           for m, b, o, tag in zip(msgs, batch, offs, tags)]
    rng = np.random.default_rng(4004)
    with_aad = [i for i, m in enumerate(msgs) if m.aad.size]
    f_ct, f_tag, f_aad = int(rng.integers(0, 10000)), int(rng.integers(0, 10000)), with_aad[int(rng.integers(0, len(with_aad)))]
    assert len({f_ct, f_tag, f_aad}) == 3
    d_out[offs[f_ct] + int(rng.integers(0, msgs[f_ct].payload.size))] ^= 0x80
    dec[f_tag]["tag"] = bytes([dec[f_tag]["tag"][0] ^ 1]) + dec[f_tag]["tag"][1:]
    forged = d_aad[aoffs[f_aad]: aoffs[f_aad] + msgs[f_aad].aad.size].clone()
    forged[0] ^= 2
    dec[f_aad]["aad"] = forged
    st = G.gcm_decrypt_verify_batch(dec)
    back = d_back.cpu().numpy()
    for i, (m, o) in enumerate(zip(msgs, offs)):
        if i in (f_ct, f_tag, f_aad):
            assert st[i] == G.GCM_ERR_AUTH, m.name
            assert not back[o: o + m.payload.size].any(), m.name
        else:
            assert st[i] == G.GCM_OK, m.name
            assert np.array_equal(back[o: o + m.payload.size], m.payload), m.name
    G.gcm_batch_release()


def test_config_c5_full(G, oracle):
    """C5: AES-256-GCM, one 4 GiB message (the bench.py workload: payload generated on the device from
    the config's seed, 2880-byte header AAD), encrypt, decrypt_verify, and a copy with one seeded
    ciphertext bit flipped that must be rejected with an all-zero output."""
    free, _ = torch.cuda.mem_get_info()
    if free < 14 << 30:
        pytest.skip("needs 14 GiB of free device memory")
    n = 4 << 30
    m = workloads.config_c5(payload_bytes=n, with_payload=False)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(workloads.SEEDS["C5"])
    d_pt = torch.randint(-2 ** 63, 2 ** 63 - 1, (n // 8,), dtype=torch.int64, device="cuda", generator=gen).view(torch.uint8)
    d_ct = torch.empty(n, dtype=torch.uint8, device="cuda")
    d_aad = dev(m.aad)
    ctx = G.gcm_init(m.key)
    try:
        assert G.gcm_get_geometry(ctx) == (torch.cuda.get_device_properties(0).multi_processor_count, 512)
        tag = G.gcm_encrypt(ctx, m.iv, d_aad, d_pt, d_ct)
        oracle_check_device_message(oracle, m.key, m.iv, m.aad, d_pt, d_ct, tag, "C5")
        d_back = torch.empty(n, dtype=torch.uint8, device="cuda")
        assert G.gcm_decrypt_verify(ctx, m.iv, d_aad, d_ct, d_back, tag) == G.GCM_OK
        assert torch.equal(d_back, d_pt)
        bit = m.meta["flip_bit"]
        d_ct[bit // 8] ^= (1 << (bit % 8))
        assert G.gcm_decrypt_verify(ctx, m.iv, d_aad, d_ct, d_back, tag) == G.GCM_ERR_AUTH
        assert not bool(d_back.any().item())
    finally:
        G.gcm_destroy(ctx)


def test_beyond_4gib_ragged(G, oracle):
    """Maximum-size edge of the single-message path that C5 does not reach: byte offsets above 2^32 and block
    indices above 2^28 (64-bit offsets, 32-bit counters), with a ragged 13-byte tail.  Every ciphertext byte and
    the tag against the oracle, then the round trip."""
    free, _ = torch.cuda.mem_get_info()
    if free < 14 << 30:
        pytest.skip("needs 14 GiB of free device memory")
    n = (4 << 30) + (32 << 20) + 13
    m = workloads.config_c5(payload_bytes=16, with_payload=False)     # key, IV and header AAD of the C5 recipe
    gen = torch.Generator(device="cuda")
    gen.manual_seed(77)
    d_pt = torch.randint(-2 ** 63, 2 ** 63 - 1, ((n + 7) // 8,), dtype=torch.int64, device="cuda", generator=gen).view(torch.uint8)[:n]
    d_ct = torch.empty(n, dtype=torch.uint8, device="cuda")
    d_aad = dev(m.aad[:777])                                   # AAD that is not a whole number of blocks
    ctx = G.gcm_init(m.key)
    try:
        tag = G.gcm_encrypt(ctx, m.iv, d_aad, d_pt, d_ct)
        oracle_check_device_message(oracle, m.key, m.iv, m.aad[:777], d_pt, d_ct, tag, "4 GiB + 32 MiB + 13")
        d_back = torch.empty(n, dtype=torch.uint8, device="cuda")
        assert G.gcm_decrypt_verify(ctx, m.iv, d_aad, d_ct, d_back, tag) == G.GCM_OK
        assert torch.equal(d_back, d_pt)
        d_ct[n - 1] ^= 0x40                                    # last (partial-block) byte, above 2^32
        assert G.gcm_decrypt_verify(ctx, m.iv, d_aad, d_ct, d_back, tag) == G.GCM_ERR_AUTH
        assert not bool(d_back.any().item())
    finally:
        G.gcm_destroy(ctx)
