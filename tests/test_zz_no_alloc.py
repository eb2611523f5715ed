"""ms_exclusive_scan_static (include/mlpsplat.h): the offset scan of stages (a), (c), (d) as an entry point that
allocates nothing -- its tile sums live in a fixed file-scope device array -- against the path the render uses
(ms_exclusive_scan_device) and against a host prefix sum.  Integer work: bit-exact.  Collected last on purpose (the
suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _api():
    from paper_2606_03877_b200 import api
    return api


def _counts(n, seed, hi=50):
    rng = np.random.default_rng(seed)
    return rng.integers(0, hi, size=n, dtype=np.int64).astype(np.int32)


def _host_scan(c):
    out = np.zeros(c.size + 1, dtype=np.uint64)
    np.cumsum(c.astype(np.uint32).astype(np.uint64), out=out[1:])
    return (out & 0xFFFFFFFF).astype(np.uint32)


# one tile, just above one tile, the range the render's path serves with one CTA, two levels of tile sums with a
# ragged tail, the maximum
SIZES = [1, 2048, 2049, 30000, 100003, (1 << 22) + 77, 1 << 24]


def test_static_scan_matches_the_render_path_on_calls_in_a_row():
    api = _api()
    out_s = torch.empty((1 << 24) + 1, dtype=torch.int32, device="cuda")
    # descending then ascending sizes: a call after a larger one finds the larger one's tile sums in the shared array
    for rep, sizes in enumerate((SIZES[::-1], SIZES)):
        for n in sizes:
            c = _counts(n, 100 * rep + n % 97)
            d = torch.from_numpy(c).cuda()
            ref = api.exclusive_scan(d)                               # existing path: cudaMalloc'ed scratch
            for call in range(2):                                     # two calls in a row, same output buffer
                out_s[: n + 1].fill_(-1)
                got = api.exclusive_scan(d, out=out_s, static=True)[: n + 1]
                torch.cuda.synchronize()
                assert torch.equal(got, ref), (n, rep, call)
            assert np.array_equal(ref.cpu().numpy().view(np.uint32), _host_scan(c)), n


def test_static_scan_wraps_like_uint32_and_handles_empty_input():
    api = _api()
    c = np.full(5000, 0x7FFFFFFF, dtype=np.int32)                     # totals far beyond 2^32
    d = torch.from_numpy(c).cuda()
    got = api.exclusive_scan(d, static=True)
    assert torch.equal(got, api.exclusive_scan(d))
    assert np.array_equal(got.cpu().numpy().view(np.uint32), _host_scan(c))
    e = torch.empty(0, dtype=torch.int32, device="cuda")
    assert api.exclusive_scan(e, static=True).tolist() == [0] == api.exclusive_scan(e).tolist()


def test_static_scan_rejects_sizes_beyond_its_array():
    api = _api()
    n = api.SCAN_STATIC_MAX + 1
    d = torch.zeros(n, dtype=torch.int32, device="cuda")
    out = torch.full((n + 1,), 7, dtype=torch.int32, device="cuda")
    with pytest.raises(api.MsError) as e:
        api.exclusive_scan(d, out=out, static=True)
    assert e.value.code == -5                                         # MS_ERR_CAPACITY
    torch.cuda.synchronize()
    assert int(out[0]) == 7 and int(out[-1]) == 7                     # nothing was enqueued
    assert int(api.exclusive_scan(d)[-1]) == 0                        # the allocating path has no such limit


def test_static_scan_runs_under_stream_capture():
    """a cudaMalloc inside a capturing stream fails the capture: the entry point must go through, and the replayed
    graph must give the scan of whatever the input buffer holds at replay time"""
    api = _api()
    n = 70001
    d = torch.from_numpy(_counts(n, 5)).cuda()
    out = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    api.exclusive_scan(d, out=out, static=True)                       # set-up call: the array's address is known
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        api.exclusive_scan(d, out=out, static=True)
    for seed in (6, 7):
        c = _counts(n, seed)
        d.copy_(torch.from_numpy(c))
        out.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), _host_scan(c))
