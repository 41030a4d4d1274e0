"""lst_scan_counts_static: the slot-offset scan for callers that are not allowed to allocate device memory.

Some users of this library run inside a trigger / reconstruction framework that owns all device memory and bans
cudaMalloc and cudaFree from its event loop (either call synchronises the whole device, so one module allocating
stalls every other stream), or call from a place where the CUDA runtime refuses allocations altogether.  For them
include/lst.h offers ONE entry point whose scratch (the tile ticket and the tile status words of the look-back
scan) is a fixed 128 KB array inside the library instead of a cudaMalloc block.  The price is a size limit
(LST_SCAN_STATIC_MAX_N counts) and one shared array per GPU: it keeps the previous call's contents, so each call
has to clear what it uses, and calls must not overlap on the GPU.

What is checked here: on consecutive calls -- a long one, then a short one that lands on the long one's leftovers,
with no synchronisation in between -- the offsets are bit-identical to those of lst_scan_counts (the chain's own
scan kernel with scratch from cudaMalloc) and to a host prefix sum; free device memory does not move across the
calls; sizes beyond the limit are refused with LST_ERR_LIMIT and write nothing.

This file is named so that pytest collects it last: with `-x` a failure here hides no other test.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lst():
    import torch

    assert torch.cuda.is_available()
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def owner_counts(n, seed):
    """Objects per owner as the chain sees them: most owners have none, some a few, a handful hundreds."""
    rng = np.random.default_rng(seed)
    c = rng.poisson(1.5, n) * (rng.random(n) < 0.2)
    heavy = rng.integers(0, max(n, 1), size=min(n, 50))
    if n:
        c[heavy] += rng.integers(100, 2000, size=heavy.size)
    return c.astype(np.int32)


def host_offsets(c):
    return np.concatenate([[0], np.cumsum(c.astype(np.int64))]).astype(np.int32)


def test_two_calls_in_a_row_match_the_allocating_path(lst):
    import torch

    dev = torch.device("cuda:0")
    torch.cuda.set_device(0)
    # 2930 tiles with a ragged tail, then 69 tiles inside the region the first call left full of status words,
    # then a single partial tile, then the first size again
    sizes = (3_000_017, 70_001, 5, 3_000_017)
    counts = [torch.from_numpy(owner_counts(n, 11 + i)).to(dev) for i, n in enumerate(sizes)]
    want = [torch.full((n + 1,), -1, dtype=torch.int32, device=dev) for n in sizes]
    for c, w in zip(counts, want):
        lst.lst_scan_counts(c, w)  # existing path: k_scan with cudaMalloc'd scratch, synchronous
    for c, w in zip(counts, want):
        assert np.array_equal(w.cpu().numpy(), host_offsets(c.cpu().numpy()))

    # a first call (it also does the once-per-device look-up of the array's address), then the measured ones
    warm = torch.empty(sizes[1] + 1, dtype=torch.int32, device=dev)
    lst.lst_scan_counts_static(counts[1], warm)
    torch.cuda.synchronize()
    assert torch.equal(warm, want[1])

    got = [torch.full((n + 1,), -1, dtype=torch.int32, device=dev) for n in sizes]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for c, g in zip(counts, got):  # back to back on one stream, nothing waits in between
        lst.lst_scan_counts_static(c, g)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the non-allocating entry point changed free device memory"
    for n, g, w in zip(sizes, got, want):
        assert torch.equal(g, w), f"n = {n}: offsets differ from lst_scan_counts"

    # the same on a stream of the caller's
    side = torch.cuda.Stream()
    got2 = [torch.full((n + 1,), -1, dtype=torch.int32, device=dev) for n in sizes]
    torch.cuda.synchronize()
    for c, g in zip(counts, got2):
        lst.lst_scan_counts_static(c, g, side.cuda_stream)
    side.synchronize()
    for n, g, w in zip(sizes, got2, want):
        assert torch.equal(g, w), f"n = {n} (side stream): offsets differ from lst_scan_counts"


def test_empty_and_largest_size(lst):
    import torch

    dev = torch.device("cuda:0")
    empty = torch.empty(0, dtype=torch.int32, device=dev)
    out = torch.full((1,), -1, dtype=torch.int32, device=dev)
    lst.lst_scan_counts_static(empty, out)
    torch.cuda.synchronize()
    assert out.item() == 0
    n = lst.LST_SCAN_STATIC_MAX_N  # every status word of the array in use
    c = torch.from_numpy(owner_counts(n, 3)).to(dev)
    want = torch.empty(n + 1, dtype=torch.int32, device=dev)
    got = torch.empty(n + 1, dtype=torch.int32, device=dev)
    lst.lst_scan_counts(c, want)
    for _ in range(2):
        got.fill_(-1)
        lst.lst_scan_counts_static(c, got)
        torch.cuda.synchronize()
        assert torch.equal(got, want)
    assert int(want[-1].item()) == int(c.sum(dtype=torch.int64).item())


def test_sizes_beyond_the_limit_are_refused(lst):
    import ctypes as C

    import torch

    from paper_2407_18231_b200 import binding

    dev = torch.device("cuda:0")
    c = torch.ones(1024, dtype=torch.int32, device=dev)
    out = torch.full((1025,), -7, dtype=torch.int32, device=dev)
    # the raw call with a length the arrays do not have: it must be turned down before anything is touched
    rc = binding._lib().lst_scan_counts_static(C.c_void_p(c.data_ptr()), lst.LST_SCAN_STATIC_MAX_N + 1,
                                               C.c_void_p(out.data_ptr()), None)
    torch.cuda.synchronize()
    assert rc == lst.LST_ERR_LIMIT
    assert "LST_SCAN_STATIC_MAX_N" in binding._lib().lst_strerror(rc).decode()
    assert bool((out == -7).all())
    with pytest.raises(lst.LstError) as e:
        lst.lst_scan_counts_static(torch.ones(lst.LST_SCAN_STATIC_MAX_N + 1, dtype=torch.int32, device=dev),
                                   torch.empty(lst.LST_SCAN_STATIC_MAX_N + 2, dtype=torch.int32, device=dev))
    assert e.value.status == lst.LST_ERR_LIMIT
