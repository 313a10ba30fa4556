"""splotch_scan_static: the bin-offset scan for callers that may not allocate device memory.

Some programs that embed this library cannot call cudaMalloc and have no spare device buffer to lend: a renderer
running in situ inside a simulation whose own pool owns all of the GPU's memory is the typical case (an allocation
by a plug-in could fail, could starve the simulation's next step, and stalls every stream of the device while it
runs).  splotch_scan_static serves them: its tile bookkeeping sits in a fixed 66,048-byte array inside the library,
so the caller passes only its input counts and its output offsets.

What is checked here: the offsets are bit for bit those of the existing path (splotch_debug_scan with scratch the
caller allocated; the bar for integer work is exact equality) on two calls in a row, the second one smaller and on
different data, so that anything the first call left in the shared array would show; the stated size limit is
enforced with SPLOTCH_ERR_LIMIT; and n = 0 works.  The file sorts last on purpose (pytest -x stops at the first
failure, and a failure here must not hide the parity tests), and it passes both alone in a fresh process, where its
first call is the one that looks up the array's device address, and after the other GPU tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1004_1302_b200 import binding
    binding.library_path()
    return binding


def _counts(n, seed):
    rs = np.random.RandomState(seed)
    return rs.randint(0, 2 ** 32, size=max(n, 1), dtype=np.uint64).astype(np.uint32)[:n]


def _device_counts(a):
    d = torch.zeros(max(a.size, 1), dtype=torch.int32, device="cuda")
    if a.size:
        d[: a.size] = torch.from_numpy(a.view(np.int32)).cuda()
    return d


def _existing_path(B, d_in, n):
    """The scan as the rest of the library calls it: scratch allocated by the caller."""
    out = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
    sb = (n // 2048 + 2) * 8 + 512
    scratch = torch.empty(sb, dtype=torch.uint8, device="cuda")
    B.splotch_debug_scan(d_in, out, n, scratch, sb)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint64)


def test_static_scan_equals_existing_scan_on_two_calls_in_a_row(B):
    # first call: many tiles and a ragged tail; second call: fewer tiles, other data, same shared array
    cases = [(1_000_003, 11), (300_001, 12)]
    inputs = [(n, _counts(n, seed)) for n, seed in cases]
    d_ins = [_device_counts(a) for _, a in inputs]
    # outputs pre-filled with a pattern, so an element the kernel did not write cannot pass by accident
    outs = [torch.full((n + 1,), -1, dtype=torch.int64, device="cuda") for n, _ in inputs]
    for (n, _), d_in, out in zip(inputs, d_ins, outs):          # back to back on one stream, no sync in between
        B.splotch_scan_static(d_in, out, n)
    torch.cuda.synchronize()
    for (n, a), d_in, out in zip(inputs, d_ins, outs):
        got = out.cpu().numpy().view(np.uint64)
        np.testing.assert_array_equal(got, _existing_path(B, d_in, n))
        assert got[0] == 0 and got[n] == a.astype(np.uint64).sum()          # sums overflow 32 bits: 64-bit offsets


def test_static_scan_edge_sizes_and_limit(B):
    for n in (0, 1, 2048, 2049):
        a = _counts(n, 20 + n)
        d_in = _device_counts(a)
        out = torch.full((n + 1,), -1, dtype=torch.int64, device="cuda")
        B.splotch_scan_static(d_in if n else None, out, n)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(out.cpu().numpy().view(np.uint64), _existing_path(B, d_in, n))
    # one past the limit: refused before anything is enqueued, output untouched
    n = B.SPLOTCH_SCAN_STATIC_MAX_N + 1
    d_in = torch.zeros(8, dtype=torch.int32, device="cuda")
    out = torch.full((8,), -1, dtype=torch.int64, device="cuda")
    with pytest.raises(B.SplotchError) as e:
        B.splotch_scan_static(d_in, out, n)
    assert e.value.status == B.SPLOTCH_ERR_LIMIT
    torch.cuda.synchronize()
    assert bool((out == -1).all())
    with pytest.raises(B.SplotchError) as e:
        B.splotch_scan_static(d_in, None, 8)
    assert e.value.status == B.SPLOTCH_ERR_INVALID_ARG


def test_static_scan_at_the_limit(B):
    n = B.SPLOTCH_SCAN_STATIC_MAX_N                                   # all 8192 tiles, every descriptor in use
    a = _counts(n, 31)
    d_in = _device_counts(a)
    out = torch.full((n + 1,), -1, dtype=torch.int64, device="cuda")
    B.splotch_scan_static(d_in, out, n)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(out.cpu().numpy().view(np.uint64), _existing_path(B, d_in, n))
