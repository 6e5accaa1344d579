"""gfc_datasum_noalloc (include/gfc.h): the DATASUM entry point for callers that cannot allocate device memory.

Who needs it: a program in which the GPU's memory already belongs to someone else (a caching allocator or a
pre-reserved pool holds all of it, so the cudaMalloc inside gfc_datasum would fail), and a program that calls
the checksum in a latency-critical loop next to other streams (cudaMalloc / cudaFree can make the whole device
wait).  The entry point keeps its scratch (one partial sum per 256 KiB tile and a ticket counter) in a fixed
128.25 KiB array inside the library's device image and allocates nothing.

What is checked: its result equals the result of the existing path, gfc_datasum, bit for bit (the bar every
integer test of this suite uses), on several calls IN A ROW -- the array is shared by all calls and keeps what
the previous call left in it, so a long buffer followed by a short one, and the same buffer twice, would show
stale partials or a ticket counter that did not start at zero.  The existing path is itself held against the
oracle's sum in test_gpu_frame.py::test_datasum_kernel; one case here repeats that check directly.

This file is named so that pytest collects it last (`pytest --collect-only -q`): under `pytest -x` a failure here
cannot hide the result of any other test.  It passes on its own in a fresh process (then its first call is the
one that looks up the scratch's address and loads the module on the device) and after the other GPU tests.
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gfc():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2602_23067_b200 import gfc as g
    return g


def _buffers(sizes, seed):
    import torch
    rng = np.random.default_rng(seed)
    out = []
    for n in sizes:
        a = rng.integers(0, 256, n, dtype=np.uint8)
        if n >= 2880:
            a[: n // 2] = 0xFF                      # long runs of end-around carries
        out.append((a, torch.from_numpy(a).cuda()))
    return out


def _noalloc(gfc, d, d_sum):
    import torch
    d_sum.fill_(-1)                                 # a call that wrote nothing would be seen
    gfc.gfc_datasum_noalloc(d, d_sum)
    torch.cuda.synchronize()
    return int(d_sum.item()) & 0xFFFFFFFF


TILE = 256 << 10


def test_two_calls_in_a_row_match_the_existing_path(gfc):
    """A long buffer (193 tiles, ragged), then a short one (3 tiles) that must not see the long one's partials,
    then the first again: each equal to gfc_datasum of the same buffer."""
    import torch
    bufs = _buffers([(48 << 20) + 16 * 3 + 2, 2 * TILE + 2880 * 7 + 5, 13], seed=31)
    want = [gfc.gfc_datasum(d) for _, d in bufs]
    d_sum = torch.zeros(1, dtype=torch.int32, device="cuda")
    got = [_noalloc(gfc, d, d_sum) for _, d in bufs]                     # calls back to back on one stream
    assert got == want
    assert _noalloc(gfc, bufs[0][1], d_sum) == want[0]                   # after the short ones
    assert _noalloc(gfc, bufs[0][1], d_sum) == want[0]                   # and the same call twice


def test_back_to_back_without_a_host_wait_between(gfc):
    """Two calls enqueued on one stream with no synchronisation between them (stream order is the only thing that
    separates their use of the shared scratch), each into its own output word."""
    import torch
    (_, d0), (_, d1) = _buffers([5 * TILE + 17, 9 * TILE], seed=32)
    want = [gfc.gfc_datasum(d0), gfc.gfc_datasum(d1)]
    sums = torch.full((2,), -1, dtype=torch.int32, device="cuda")
    gfc.gfc_datasum_noalloc(d0, sums[0:1])
    gfc.gfc_datasum_noalloc(d1, sums[1:2])
    torch.cuda.synchronize()
    assert [int(v) & 0xFFFFFFFF for v in sums.tolist()] == want


def test_tile_edges_and_empty(gfc):
    import torch
    from oracle import fits_container as F
    sizes = [0, 1, 3, 4, 15, 16, 17, 2880, TILE - 16, TILE - 1, TILE, TILE + 1, TILE + 16, 4 * TILE + 15]
    d_sum = torch.zeros(1, dtype=torch.int32, device="cuda")
    for a, d in _buffers(sizes, seed=33):
        n = a.size
        got = _noalloc(gfc, d, d_sum)
        assert got == gfc.gfc_datasum(d), n
        assert got == F.sum32(a.tobytes() + b"\0" * ((-n) % 4)), n       # and the oracle's sum directly


def test_sizes_beyond_the_scratch_are_refused(gfc):
    """More than 4 GiB would need more partials than the array holds: GCM_ERR_LEN before anything is enqueued (the
    call is made with a small buffer's address and a large length, so a launch would fault)."""
    import torch
    from paper_2602_23067_b200 import gcm
    d = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    d_sum = torch.full((1,), 7, dtype=torch.int32, device="cuda")
    big = gfc.GFC_DATASUM_NOALLOC_MAX_BYTES + 1
    with pytest.raises(gcm.GcmError) as e:
        gfc.gfc_datasum_noalloc((d.data_ptr(), big), d_sum)
    assert e.value.code == gcm.GCM_ERR_LEN
    torch.cuda.synchronize()
    assert int(d_sum.item()) == 7                                        # untouched
    L = gfc._L
    assert L.gfc_datasum_noalloc(d.data_ptr(), 16, None, None) == gcm.GCM_ERR_ARG
    assert L.gfc_datasum_noalloc(d.data_ptr() + 4, 16, d_sum.data_ptr(), None) == gcm.GCM_ERR_ARG
    assert L.gfc_datasum_noalloc(None, 16, d_sum.data_ptr(), None) == gcm.GCM_ERR_ARG
    assert _noalloc(gfc, d, d_sum) == 0                                  # still usable afterwards


def test_full_size_limit(gfc):
    """Exactly 4 GiB: all 16384 partials in use."""
    import torch
    n = gfc.GFC_DATASUM_NOALLOC_MAX_BYTES
    free, _ = torch.cuda.mem_get_info()
    if free < n + (1 << 30):
        pytest.skip("not enough free device memory for a 4 GiB buffer")
    d = torch.empty(n, dtype=torch.uint8, device="cuda")
    g = torch.Generator(device="cuda").manual_seed(34)
    d.view(torch.int64).random_(generator=g)
    d_sum = torch.zeros(1, dtype=torch.int32, device="cuda")
    want = gfc.gfc_datasum(d)
    assert _noalloc(gfc, d, d_sum) == want
    assert _noalloc(gfc, d[: n - 3 * TILE - 16], d_sum) == gfc.gfc_datasum(d[: n - 3 * TILE - 16])
    del d
    torch.cuda.empty_cache()
