"""Robustness of the C-ABI boundary on the GPU ("What's weak" 8): one call at a
time per context (GCM_ERR_BUSY, never a race), verdicts that fail closed, verify-then-release for host buffers
(PAPER.md L45, L93, L219), the caller's current device left alone, the phase-stamp diagnostics."""
import threading

import numpy as np
import pytest

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


def test_strict_host_decrypt_releases_nothing_unverified(G, oracle):
    """gcm_decrypt_verify_host_strict: GHASH-only pass first, decrypt only after the tag matched.  On a forged
    message the caller's buffer is not touched at all (not even zero-filled); on a good one it equals the oracle's
    plaintext.  Sizes: empty, one chunk, several chunks with a ragged tail."""
    rng = np.random.default_rng(9950)
    key = rnd(rng, 32).tobytes()
    ctx = G.gcm_init(key)
    try:
        for (n, a) in [(0, 0), (0, 33), (1, 0), (100003, 2880), ((40 << 20) + 777, 17)]:
            iv = rnd(rng, 12).tobytes()
            aad = rnd(rng, a)
            pt = rnd(rng, n)
            ct, tag = oracle.gcm_encrypt_threaded(key, iv, aad, pt, threads=8, segment_blocks=1 << 16) if n > (1 << 20) \
                else oracle.gcm_encrypt(key, iv, aad, pt)
            h_ct = torch.from_numpy(ct.copy()).pin_memory()
            back = torch.full((n,), 0x5A, dtype=torch.uint8).pin_memory()
            assert G.gcm_decrypt_verify_host_strict(ctx, iv, aad, h_ct, back, tag) == G.GCM_OK, (n, a)
            assert np.array_equal(back.numpy(), pt), (n, a)
            # forged: tag, and (when there is one) a ciphertext byte, an AAD byte
            forgeries = [dict(tag=bytes([tag[0] ^ 1]) + tag[1:])]
            if n:
                bad = h_ct.clone(); bad[n - 1] ^= 0x80
                forgeries.append(dict(ct=bad))
            if a:
                bad_aad = aad.copy(); bad_aad[a // 2] ^= 4
                forgeries.append(dict(aad=bad_aad))
            for f in forgeries:
                back.fill_(0x5A)
                rc = G.gcm_decrypt_verify_host_strict(ctx, iv, f.get("aad", aad), f.get("ct", h_ct), back, f.get("tag", tag))
                assert rc == G.GCM_ERR_AUTH, (n, a, list(f))
                assert bool((back == 0x5A).all().item()), "unverified bytes reached the caller's buffer"
            # the non-strict form on the same forgery: refused and zero-filled
            if n:
                back.fill_(0x5A)
                assert G.gcm_decrypt_verify_host(ctx, iv, aad, forgeries[1]["ct"], back, tag) == G.GCM_ERR_AUTH
                assert not bool(back.any().item())
    finally:
        G.gcm_destroy(ctx)


def test_one_call_at_a_time_per_context(G, oracle):
    """Two host threads on ONE context: a call that finds the context in use returns GCM_ERR_BUSY and does nothing;
    every call that does run returns the oracle's tag (no silent race on the cross-CTA scratch)."""
    rng = np.random.default_rng(9960)
    key = rnd(rng, 16).tobytes()
    iv = rnd(rng, 12).tobytes()
    big = rnd(rng, 96 << 20)
    small = rnd(rng, 16 * 512 * 9 + 3)
    ref_big = oracle.gcm_encrypt_threaded(key, iv, b"", big, threads=8, segment_blocks=1 << 16)[1]
    ref_small = oracle.gcm_encrypt(key, iv, b"", small)[1]
    ctx = G.gcm_init(key)
    h_in = torch.from_numpy(big).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    d_small, d_out = dev(small), torch.empty(small.size, dtype=torch.uint8, device="cuda")
    s2 = torch.cuda.Stream()
    stop = threading.Event()
    seen = {"busy": 0, "ok": 0, "bad": 0, "big_ok": 0, "big_busy": 0, "big_bad": 0}

    def long_calls():
        for _ in range(6):
            try:
                t = G.gcm_encrypt_host(ctx, iv, None, h_in, h_out)          # several ms inside the library
                seen["big_ok" if t == ref_big else "big_bad"] += 1
            except G.GcmError as e:
                seen["big_busy" if e.code == G.GCM_ERR_BUSY else "big_bad"] += 1
        stop.set()

    th = threading.Thread(target=long_calls)
    try:
        th.start()
        while not stop.is_set():
            try:
                t = G.gcm_encrypt(ctx, iv, None, d_small, d_out, s2)
                seen["ok" if t == ref_small else "bad"] += 1
            except G.GcmError as e:
                seen["busy" if e.code == G.GCM_ERR_BUSY else "bad"] += 1
        th.join()
        assert seen["bad"] == 0 and seen["big_bad"] == 0, seen
        assert seen["busy"] > 0, "the second thread never met the busy context: %r" % seen
        assert seen["big_ok"] + seen["big_busy"] == 6 and seen["big_ok"] > 0, seen
        # the context is fine afterwards
        assert G.gcm_encrypt(ctx, iv, None, d_small, d_out) == ref_small
    finally:
        th.join()
        G.gcm_destroy(ctx)


def test_async_verdict_fails_closed_and_is_rewritten_every_call(G, oracle):
    """The device verdict word is set to a refusing value by the launch itself before the finisher writes it: a
    stale 0 (accepted) from an earlier call can never stand for this one."""
    rng = np.random.default_rng(9970)
    key = rnd(rng, 32).tobytes()
    iv = rnd(rng, 12).tobytes()
    pt = rnd(rng, 16 * 512 * 20 + 1)
    ct, tag = oracle.gcm_encrypt(key, iv, b"", pt)
    ctx = G.gcm_init(key)
    try:
        d_ct, d_tag = dev(ct), dev(np.frombuffer(tag, np.uint8))
        out = torch.empty(pt.size, dtype=torch.uint8, device="cuda")
        d_status = torch.zeros(1, dtype=torch.int32, device="cuda")           # stale "accepted"
        bad = d_ct.clone(); bad[17] ^= 1
        for geometry in [(0, 0), (3, 256), (148, 384)]:
            G.gcm_set_geometry(ctx, *geometry)
            d_status.zero_()
            G.gcm_decrypt_verify_async(ctx, iv, None, bad, out, d_tag, d_status)
            torch.cuda.synchronize()
            assert int(d_status.item()) == G.GCM_ERR_AUTH and not bool(out.any().item()), geometry
            d_status.fill_(1)                                                   # stale "refused"
            G.gcm_decrypt_verify_async(ctx, iv, None, d_ct, out, d_tag, d_status)
            torch.cuda.synchronize()
            assert int(d_status.item()) == G.GCM_OK and np.array_equal(out.cpu().numpy(), pt), geometry
    finally:
        G.gcm_destroy(ctx)


@pytest.mark.parametrize("n", [1, 100, 16 * 509, 8000])
def test_async_verdict_of_header_sized_messages(G, oracle, n):
    """The same contract for messages of at most 511 GHASH blocks, which the default geometry sends to the one-CTA
    latency kernel (gcm_small.cu): that kernel too overwrites a stale verdict, in both directions."""
    rng = np.random.default_rng(9980 + n)
    for key_bytes in (16, 32):
        key, iv, aad = rnd(rng, key_bytes).tobytes(), rnd(rng, 12).tobytes(), rnd(rng, 21).tobytes()
        pt = rnd(rng, n)
        ct, tag = oracle.gcm_encrypt(key, iv, aad, pt)
        ctx = G.gcm_init(key)
        try:
            d_ct, d_tag, d_aad = dev(ct), dev(np.frombuffer(tag, np.uint8)), dev(np.frombuffer(aad, np.uint8))
            out = torch.full((n,), 0xAA, dtype=torch.uint8, device="cuda")
            d_status = torch.zeros(1, dtype=torch.int32, device="cuda")       # stale "accepted"
            bad = d_ct.clone(); bad[n // 2] ^= 0x80
            G.gcm_decrypt_verify_async(ctx, iv, d_aad, bad, out, d_tag, d_status)
            torch.cuda.synchronize()
            assert int(d_status.item()) == G.GCM_ERR_AUTH and not bool(out.any().item())
            d_status.fill_(1)                                                   # stale "refused"
            G.gcm_decrypt_verify_async(ctx, iv, d_aad, d_ct, out, d_tag, d_status)
            torch.cuda.synchronize()
            assert int(d_status.item()) == G.GCM_OK and np.array_equal(out.cpu().numpy(), pt)
        finally:
            G.gcm_destroy(ctx)


def test_device_selection_and_current_device_untouched(G):
    """gcm_set_device only records the ordinal; contexts live on it (or on the caller's current device); no call
    changes the calling thread's current CUDA device."""
    import ctypes
    from paper_2602_23067_b200 import gcm as B
    before = torch.cuda.current_device()
    assert B._L.gcm_set_device(torch.cuda.device_count() + 3) == G.GCM_ERR_ARG
    G.gcm_set_device(-1)                          # back to "the caller's current device"
    ctx = G.gcm_init(bytes(16))
    try:
        t = torch.zeros(4096, dtype=torch.uint8, device="cuda")
        G.gcm_encrypt(ctx, bytes(12), None, t, t)
        assert torch.cuda.current_device() == before
        G.gcm_set_device(0)
        ctx2 = G.gcm_init(bytes(32))
        G.gcm_encrypt(ctx2, bytes(12), None, t, t)
        G.gcm_destroy(ctx2)
        assert torch.cuda.current_device() == before
    finally:
        G.gcm_destroy(ctx)
        G.gcm_set_device(-1)


def test_phase_stamps(G):
    """gcm_set_phase_stamps: one record of %globaltimer values per CTA, non-decreasing along the kernel's phases,
    and no effect on the result."""
    ctx = G.gcm_init(bytes(range(32)))
    try:
        grid, _ = G.gcm_get_geometry(ctx)
        n = 8 << 20
        pt = torch.arange(n, dtype=torch.int64, device="cuda").to(torch.uint8)
        ct1, ct2 = torch.empty_like(pt), torch.empty_like(pt)
        tag1 = G.gcm_encrypt(ctx, bytes(12), None, pt, ct1)
        stamps = torch.zeros(G.GCM_PHASE_SLOTS * grid, dtype=torch.int64, device="cuda")
        G.gcm_set_phase_stamps(ctx, stamps)
        tag2 = G.gcm_encrypt(ctx, bytes(12), None, pt, ct2)
        G.gcm_set_phase_stamps(ctx, None)
        assert tag1 == tag2 and torch.equal(ct1, ct2)
        st = stamps.cpu().numpy().reshape(grid, G.GCM_PHASE_SLOTS)
        live = st[st[:, 0] > 0]
        assert live.shape[0] == grid
        assert (np.diff(live[:, :6], axis=1) >= 0).all()
        assert (live[:, 6] > 0).sum() == 1                    # exactly one CTA finished the message
    finally:
        G.gcm_destroy(ctx)

