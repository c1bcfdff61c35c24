"""tcrnet_row_ptr_noalloc (include/tcrnet.h): the prefix-sum step of A6 with its scratch in a static device array, for
callers that cannot allocate.  Its output is compared, bit for bit (integers), with the row_ptr the existing path
(tcrnet_load + tcrnet_build, scratch from the context's allocator) produced for the same counts - on calls in a row that
share the array, the later ones smaller than the earlier ones, so whatever a call leaves behind would show.

This file sorts last on purpose: the suite runs with pytest -x, a failure here must not hide the other tests.
"""
import numpy as np
import pytest

from cdr3_synth import generate

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2112_06613_b200 as p
    return p


def existing_path(pkg, name, l_max, n=None):
    """(counts int32[n], row_ptr int64[n + 1]) on the device: row_ptr as tcrnet_build wrote it, counts = its differences."""
    import torch
    d = generate(name) if n is None else generate(name, n=n)
    with pkg.TcrNet(0) as net:
        net.load(d.residues, d.lengths)
        net.build(l_max)
        row_ptr = net.csr()[0].clone()
    counts = (row_ptr[1:] - row_ptr[:-1]).to(torch.int32).contiguous()
    assert int(row_ptr[-1]) > 0 and row_ptr.numel() == d.n + 1
    return counts, row_ptr


def test_row_ptr_noalloc_equals_the_existing_path_on_calls_in_a_row(pkg):
    import torch
    big = existing_path(pkg, "cfg4", 1, n=pkg.NOALLOC_MAX_ROWS)  # every tile of the static array in use
    mid = existing_path(pkg, "cfg2", 2)                          # 50,000 rows: 49 tiles, ragged tail
    small = existing_path(pkg, "cfg1", 1)                        # 2,000 rows: 2 tiles
    out = {id(c): torch.full((c.numel() + 1,), -7, dtype=torch.int64, device="cuda") for c, _ in (big, mid, small)}
    # two calls in a row (and more): each later call finds the earlier ones' partial sums in the array
    for counts, want in (big, mid, small, mid, big, small, small):
        o = out[id(counts)]
        o.fill_(-7)
        pkg.row_ptr_noalloc(counts, o)
        torch.cuda.synchronize()
        assert torch.equal(o, want)
    # a caller's own stream; a prefix of a larger array (n given)
    side = torch.cuda.Stream()
    counts, want = mid
    o = out[id(counts)]
    o.fill_(-7)
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        pkg.row_ptr_noalloc(counts, o, n=12345, stream=side)
    side.synchronize()
    assert torch.equal(o[:12346], want[:12346]) and bool((o[12346:] == -7).all())


def test_row_ptr_noalloc_allocates_nothing_and_rejects_what_does_not_fit(pkg):
    import torch
    counts, want = existing_path(pkg, "cfg2", 1)
    o = torch.empty(counts.numel() + 1, dtype=torch.int64, device="cuda")
    pkg.row_ptr_noalloc(counts, o)  # (first call on the device: looks the array's address up)
    torch.cuda.synchronize()
    free0, reserved0 = torch.cuda.mem_get_info()[0], torch.cuda.memory_reserved()
    for _ in range(20):
        pkg.row_ptr_noalloc(counts, o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0 and torch.cuda.memory_reserved() == reserved0
    assert torch.equal(o, want)
    # n = 0: row_ptr[0] = 0 and nothing else
    o.fill_(5)
    pkg.row_ptr_noalloc(counts, o, n=0)
    torch.cuda.synchronize()
    assert int(o[0]) == 0 and int(o[1]) == 5
    # beyond the capacity: a clear error, nothing written, nothing launched
    o.fill_(5)
    with pytest.raises(pkg.TcrNetError) as e:
        pkg.row_ptr_noalloc(counts, o, n=pkg.NOALLOC_MAX_ROWS + 1)
    assert e.value.status == pkg.ERR_CAPACITY and "capacity" in pkg.strerror(pkg.ERR_CAPACITY)
    with pytest.raises(pkg.TcrNetError) as e:
        pkg.row_ptr_noalloc(counts, o, n=-1)
    assert e.value.status == pkg.ERR_ARG
    torch.cuda.synchronize()
    assert bool((o == 5).all())
    # and the next call is fine
    pkg.row_ptr_noalloc(counts, o)
    torch.cuda.synchronize()
    assert torch.equal(o, want)
    assert np.array_equal(o.cpu().numpy(), want.cpu().numpy())
