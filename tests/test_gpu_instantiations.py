"""GPU parity for every kernel instantiation the library can launch that the config tests do not reach
("Missing" 2): the large-message batch kernel `gcm_multi_kernel` with AES-128, several key
groups, ragged / unaligned / in-place messages and a call that mixes it with the warp-per-message kernel;
GHASH-only (`gcm_ghash_async`, Table 5 scope L363) over empty, ragged and long inputs under two
geometries.  Bar: every ciphertext byte and every tag byte equal to the oracle's (integer work, bit-exact).
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

THREADS = os.cpu_count() or 1
LARGE = 256 << 10          # BATCH_LARGE_BYTES of csrc/gcm_batch.cu: at and above, the multi-message kernel


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


def build_batch(specs):
    """specs: (key, iv, aad, pt, in_off, out_off, in_place).  Every message gets its own guarded buffers with the
    requested misalignment; returns (batch dicts, backing output tensors, offsets)."""
    batch, outs = [], []
    for (key, iv, aad, pt, oi, oo, in_place) in specs:
        n = len(pt)
        big_in = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
        big_in[oi: oi + n] = dev(pt)
        if in_place:
            big_out, oo = big_in, oi
        else:
            big_out = torch.zeros(n + 64, dtype=torch.uint8, device="cuda")
        batch.append({"key": key, "iv": iv, "aad": dev(aad) if len(aad) else None,
                      "input": big_in[oi: oi + n], "output": big_out[oo: oo + n]})
        outs.append((big_out, oo, n, in_place))
    return batch, outs


def test_batch_large_path_every_instantiation(G, oracle):
    """One gcm_encrypt_batch call that holds: three AES-128 key groups and two AES-256 key groups of large
    messages (gcm_multi_kernel<10,...> and <14,...>, one launch per key), ragged lengths (partial last block,
    partial last row), unaligned input / output / AAD (the kernel's byte-granular slow path), an in-place message,
    and small messages of both key sizes in the same call (gcm_batch_kernel).  Then gcm_decrypt_verify_batch with
    one forged message per key group: rejected and zero-filled, every neighbour intact."""
    rng = np.random.default_rng(9900)
    keys128 = [rnd(rng, 16).tobytes() for _ in range(3)]
    keys256 = [rnd(rng, 32).tobytes() for _ in range(2)]
    specs = []

    def add(key, n, a, oi=0, oo=0, in_place=False):
        specs.append((key, rnd(rng, 12).tobytes(), rnd(rng, a), rnd(rng, n), oi, oo, in_place))

    # large, AES-128, three keys
    add(keys128[0], LARGE, 0)                                   # exactly at the threshold, no AAD
    add(keys128[0], LARGE + 16 * 32 * 5 + 16 * 7 + 3, 2880)     # ragged row and ragged block
    add(keys128[0], 1 << 20, 17, oi=3)                          # unaligned input
    add(keys128[1], (1 << 20) + 1, 16, oo=5)                    # unaligned output
    add(keys128[1], 3 * LARGE + 4095, 100, oi=9, oo=9)          # both unaligned by the same amount
    add(keys128[2], 2 * LARGE + 15, 256, in_place=True)         # in place
    add(keys128[2], LARGE + 512, 1, oi=1, oo=2)
    # large, AES-256, two keys
    add(keys256[0], (1 << 21) + 13, 2880)
    add(keys256[0], LARGE + 1, 0, oi=15, oo=1)
    add(keys256[1], LARGE * 2, 33, in_place=True)
    add(keys256[1], LARGE + 16 * 31, 15)
    # small messages of both key sizes in the same call (warp-per-message kernel), one just below the threshold
    add(keys128[0], LARGE - 1, 40)
    add(rnd(rng, 16).tobytes(), 1000, 0)
    add(keys256[1], 65536 + 7, 256, oi=3, oo=3)
    add(rnd(rng, 32).tobytes(), 0, 5)
    add(rnd(rng, 16).tobytes(), 1, 0)

    batch, outs = build_batch(specs)
    refs = [oracle.gcm_encrypt(key, iv, aad, pt) for (key, iv, aad, pt, *_rest) in specs]
    tags = G.gcm_encrypt_batch(batch)
    for i, ((big_out, oo, n, in_place), (ref_ct, ref_tag), tag) in enumerate(zip(outs, refs, tags)):
        out = big_out.cpu().numpy()
        assert tag == ref_tag, "tag of message %d (len %d)" % (i, n)
        assert np.array_equal(out[oo: oo + n], ref_ct), "ciphertext of message %d (len %d)" % (i, n)
        assert not out[:oo].any() and not out[oo + n:].any(), "message %d wrote outside its output range" % i

    # decrypt_verify: one forgery per large key group (ciphertext first / middle / last byte, tag, AAD), one small
    dec, dec_outs = [], []
    for i, (b, (big_out, oo, n, _), tag) in enumerate(zip(batch, outs, tags)):
        ct = big_out[oo: oo + n].clone()
        back = torch.full((n + 32,), 0x77, dtype=torch.uint8, device="cuda")
        dec.append({"key": b["key"], "iv": b["iv"], "aad": b["aad"], "input": ct, "output": back[16: 16 + n], "tag": tag})
        dec_outs.append(back)
    bad = {1, 4, 6, 7, 10, 13}
    dec[1]["input"][0] ^= 1                                             # keys128[0]: first ciphertext byte
    dec[4]["input"][len(specs[4][3]) - 1] ^= 0x80                       # keys128[1]: last byte of an unaligned message
    t = bytearray(tags[6]); t[0] ^= 4; dec[6]["tag"] = bytes(t)         # keys128[2]: tag
    a7 = dec[7]["aad"].clone(); a7[2879] ^= 1; dec[7]["aad"] = a7       # keys256[0]: AAD
    dec[10]["input"][len(specs[10][3]) // 2] ^= 0x20                    # keys256[1]: middle byte
    dec[13]["input"][5] ^= 2                                            # a small message in the same call
    st = G.gcm_decrypt_verify_batch(dec)
    for i, (spec, back) in enumerate(zip(specs, dec_outs)):
        n = len(spec[3])
        got = back.cpu().numpy()
        assert (got[:16] == 0x77).all() and (got[16 + n:] == 0x77).all(), "message %d: guard overwritten" % i
        if i in bad:
            assert st[i] == G.GCM_ERR_AUTH, i
            assert not got[16: 16 + n].any(), "message %d not suppressed" % i
        else:
            assert st[i] == G.GCM_OK, i
            assert np.array_equal(got[16: 16 + n], spec[3]), i
    G.gcm_batch_release()


def test_batch_only_large_aes128_many_messages(G, oracle):
    """AES-128 through gcm_multi_kernel alone: 20 messages of one key whose rows are dealt across warps so that
    chunks straddle message boundaries (a warp finishes one message and starts the next)."""
    rng = np.random.default_rng(9910)
    key = rnd(rng, 16).tobytes()
    specs = []
    for i in range(20):
        n = LARGE + int(rng.integers(0, 3 * LARGE)) + (0 if i % 4 == 0 else int(rng.integers(1, 16)))
        specs.append((key, rnd(rng, 12).tobytes(), rnd(rng, [0, 16, 2880, 7][i % 4]), rnd(rng, n), 0, 0, False))
    batch, outs = build_batch(specs)
    tags = G.gcm_encrypt_batch(batch)
    for i, ((big_out, oo, n, _), spec, tag) in enumerate(zip(outs, specs, tags)):
        ref_ct, ref_tag = oracle.gcm_encrypt(spec[0], spec[1], spec[2], spec[3])
        assert tag == ref_tag, i
        assert np.array_equal(big_out[oo: oo + n].cpu().numpy(), ref_ct), i
    G.gcm_batch_release()


def test_batch_packed_once_submitted_twice(G, oracle):
    """gcm_pack_msgs: the gcm_msg array is built once and handed to the C call as is; submitting it a second time after
    the inputs changed must encrypt the new inputs (the array holds pointers, not data), and a batch packed for one
    direction is refused by the other."""
    rng = np.random.default_rng(9911)
    specs = [(rnd(rng, 16 + 16 * (i % 2)).tobytes(), rnd(rng, 12).tobytes(), rnd(rng, 5 * i), rnd(rng, n), 0, 0, False)
             for i, n in enumerate([0, 1, 4097, LARGE + 3, 2 * LARGE])]
    batch, outs = build_batch(specs)
    packed = G.gcm_pack_msgs(batch)
    assert len(packed) == len(specs)
    for rep in range(2):
        tags = G.gcm_encrypt_batch(packed)
        for i, ((big_out, oo, n, _), spec, tag) in enumerate(zip(outs, specs, tags)):
            pt = spec[3] if rep == 0 else spec[3] ^ np.uint8(0x5A)
            ref_ct, ref_tag = oracle.gcm_encrypt(spec[0], spec[1], spec[2], pt)
            assert tag == ref_tag, (rep, i)
            assert np.array_equal(big_out[oo: oo + n].cpu().numpy(), ref_ct), (rep, i)
        for b in batch:
            b["input"] ^= 0x5A
    with pytest.raises(ValueError):
        G.gcm_decrypt_verify_batch(packed)
    G.gcm_batch_release()


@pytest.mark.parametrize("geometry", [(0, 0), (5, 256), (37, 384)])
def test_ghash_only_shapes(G, oracle, geometry):
    """gcm_ghash_async (MODE_GHASH) on (a, len) in {0, 1, 16, 17, 2880} x {0, 1, 15, 16, 8191, 16*512*5+9}: empty A,
    empty C, both empty, ragged ends; default geometry and two explicit ones; AES-128 and AES-256 keys (H differs)."""
    rng = np.random.default_rng(9920)
    for klen in (16, 32):
        key = rnd(rng, klen).tobytes()
        h = oracle.hash_subkey(key)
        ctx = G.gcm_init(key)
        try:
            G.gcm_set_geometry(ctx, *geometry)
            for a in (0, 1, 16, 17, 2880):
                for n in (0, 1, 15, 16, 8191, 16 * 512 * 5 + 9):
                    aad, c = rnd(rng, a), rnd(rng, n)
                    d_s = torch.full((16,), 0xEE, dtype=torch.uint8, device="cuda")
                    G.gcm_ghash_async(ctx, dev(aad) if a else None, dev(c) if n else None, d_s)
                    torch.cuda.synchronize()
                    assert d_s.cpu().numpy().tobytes() == oracle.ghash(h, aad, c), (klen, a, n)
            # unaligned ciphertext pointer: the byte-granular path of the GHASH mode
            c = rnd(rng, 16 * 300 + 5)
            big = torch.zeros(c.size + 32, dtype=torch.uint8, device="cuda")
            big[7: 7 + c.size] = dev(c)
            d_s = torch.zeros(16, dtype=torch.uint8, device="cuda")
            G.gcm_ghash_async(ctx, None, big[7: 7 + c.size], d_s)
            torch.cuda.synchronize()
            assert d_s.cpu().numpy().tobytes() == oracle.ghash(h, b"", c)
        finally:
            G.gcm_destroy(ctx)


@pytest.mark.parametrize("geometry", [(0, 0), (148, 256)])
def test_ghash_only_long_ragged(G, oracle, geometry):
    """64 MiB + 13 bytes, 17-byte AAD: position weights beyond 2^22 blocks; the oracle by the segment identity that
    tests/test_oracle_full_size.py pins against OpenSSL and against the plain Horner chain."""
    rng = np.random.default_rng(9930)
    key = rnd(rng, 32).tobytes()
    n = (64 << 20) + 13
    aad = rnd(rng, 17)
    import workloads
    c = workloads.random_payload(rng, n)
    h = oracle.hash_subkey(key)
    ctx = G.gcm_init(key)
    try:
        G.gcm_set_geometry(ctx, *geometry)
        d_s = torch.zeros(16, dtype=torch.uint8, device="cuda")
        G.gcm_ghash_async(ctx, dev(aad), dev(c), d_s)
        torch.cuda.synchronize()
        assert d_s.cpu().numpy().tobytes() == oracle.ghash_segmented(h, aad, c, 1 << 16, THREADS)
    finally:
        G.gcm_destroy(ctx)


def test_batch_device_descriptors(G, oracle):
    """gcm_encrypt_batch_device / gcm_decrypt_verify_batch_device: descriptors resident on the device, ordering done
    by a kernel, tags and verdicts written into the descriptors.  Both key sizes in one call, every tail shape,
    empty messages, empty AAD, unaligned buffers, a descriptor with a bad key size, the same array launched twice,
    then decryption with three forgeries: refused, zero-filled, neighbours untouched.  Byte-exact against the oracle."""
    import workloads
    rng = np.random.default_rng(9940)
    lens = [0, 1, 15, 16, 17, 31, 32, 33, 495, 496, 497, 511, 512, 513, 4096, 8191, 8192 + 5, 16 * 32 * 7 + 16 * 30 + 9,
            65536, 70001, 200000, 300000] + rng.integers(1, 65537, 60).tolist()
    specs = []
    for i, n in enumerate(lens):
        klen = 16 if i % 3 else 32
        a = [0, 1, 16, 17, 100, 256, 2880][i % 7]
        specs.append((rnd(rng, klen).tobytes(), rnd(rng, 12).tobytes(), rnd(rng, a), rnd(rng, n), i % 5 == 4))
    offs, pos = [], 0
    for (_, _, _, pt, unal) in specs:
        pos = (pos + 15) // 16 * 16 + (3 if unal else 0)
        offs.append(pos)
        pos += len(pt) + 16
    big_in = torch.zeros(pos + 16, dtype=torch.uint8, device="cuda")
    big_out = torch.zeros(pos + 16, dtype=torch.uint8, device="cuda")
    for (_, _, _, pt, _), o in zip(specs, offs):
        if len(pt):
            big_in[o: o + len(pt)] = dev(pt)
    aads = [dev(aad) if len(aad) else None for (_, _, aad, _, _) in specs]
    msgs = [{"key": key, "iv": iv, "aad": d_aad, "input": big_in[o: o + len(pt)], "output": big_out[o: o + len(pt)]}
            for (key, iv, aad, pt, _), o, d_aad in zip(specs, offs, aads)]
    host = G.gcm_pack_dmsgs(msgs)
    assert host.dtype.itemsize == G.GCM_DMSG_BYTES == 112
    bad = len(msgs) // 2
    host["key_bits"][bad] = 192                                   # not a key size of reading S1
    # descriptors the ordering kernel must refuse without touching their buffers: a length that would wrap the 32-bit
    # counter, an AAD length beyond the row layout, NULL buffers with non-zero lengths
    refused = {bad: G.GCM_ERR_ARG}
    for i, (field, value, code) in zip([3, 11, 12, 13, 15], [("len", (1 << 36) - 31, G.GCM_ERR_LEN), ("aad_len", 1 << 36, G.GCM_ERR_LEN),
                                                          ("d_in", 0, G.GCM_ERR_ARG), ("d_out", 0, G.GCM_ERR_ARG), ("d_aad", 0, G.GCM_ERR_ARG)]):
        assert len(specs[i][3]) > 0 and (field != "d_aad" or len(specs[i][2]) > 0)
        host[field][i] = value
        refused[i] = code
    d_msgs = torch.from_numpy(host.view(np.uint8).copy()).cuda()
    for _ in range(2):                                            # the same descriptor array twice
        G.gcm_encrypt_batch_device(d_msgs)
    torch.cuda.synchronize()
    res = d_msgs.cpu().numpy().view(host.dtype)
    out = big_out.cpu().numpy()
    covered = np.zeros(out.size, bool)
    refs = []
    for i, ((key, iv, aad, pt, _), o) in enumerate(zip(specs, offs)):
        ref_ct, ref_tag = oracle.gcm_encrypt(key, iv, aad, pt)
        refs.append((ref_ct, ref_tag))
        if i in refused:
            assert int(res["status"][i]) == refused[i], i
            assert not out[o: o + len(pt)].any(), "a refused descriptor was processed"
            continue
        assert int(res["status"][i]) == G.GCM_OK, i
        assert res["tag"][i].tobytes() == ref_tag, "tag len=%d aad=%d" % (len(pt), len(aad))
        assert np.array_equal(out[o: o + len(pt)], ref_ct), "ct len=%d aad=%d" % (len(pt), len(aad))
        covered[o: o + len(pt)] = True
    assert not out[~covered].any(), "wrote outside a message's output range"
    # decrypt through device descriptors: oracle ciphertext in, three forgeries
    ct_in = torch.zeros_like(big_in)
    for (ref_ct, _), o in zip(refs, offs):
        if ref_ct.size:
            ct_in[o: o + ref_ct.size] = dev(ref_ct)
    dec_out = torch.full_like(big_out, 0x77)
    dmsgs = [{"key": key, "iv": iv, "aad": d_aad, "input": ct_in[o: o + len(pt)], "output": dec_out[o: o + len(pt)], "tag": ref_tag}
             for (key, iv, aad, pt, _), o, d_aad, (_, ref_tag) in zip(specs, offs, aads, refs)]
    forged = {5, 9, 20}
    t = bytearray(dmsgs[5]["tag"]); t[15] ^= 1; dmsgs[5]["tag"] = bytes(t)
    ct_in[offs[9] + len(specs[9][3]) // 2] ^= 0x10
    a20 = dmsgs[20]["aad"].clone(); a20[0] ^= 0x80; dmsgs[20]["aad"] = a20
    d_dec = torch.from_numpy(G.gcm_pack_dmsgs(dmsgs).view(np.uint8).copy()).cuda()
    G.gcm_decrypt_verify_batch_device(d_dec)
    torch.cuda.synchronize()
    st = d_dec.cpu().numpy().view(host.dtype)["status"]
    got = dec_out.cpu().numpy()
    for i, ((key, iv, aad, pt, _), o) in enumerate(zip(specs, offs)):
        if i in forged:
            assert int(st[i]) == G.GCM_ERR_AUTH, i
            assert not got[o: o + len(pt)].any(), "message %d not suppressed" % i
        else:
            assert int(st[i]) == G.GCM_OK, i
            assert np.array_equal(got[o: o + len(pt)], pt), i
    G.gcm_batch_release()
