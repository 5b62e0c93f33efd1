"""dvx_sort_pairs_no_alloc (include/dvx.h): the step-2 radix sort with its scratch in a static device array inside the
library, for callers that may not call cudaMalloc.  Checked against the existing path (dvx_sort_pairs, scratch from the
context's allocator) bit for bit - integer work - on two calls in a row, the second smaller than the first and with an odd
number of radix passes (the result then comes back out of the static buffers), without a synchronisation in between.
This file sorts last on purpose (pytest -x: a failure here hides no other test); it passes alone in a fresh process too."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23031_b200 as dvx
    c = dvx.Context(0)
    yield c
    c.close()


def _pairs(n, bits, seed):
    rng = np.random.default_rng(seed)
    keys = rng.integers(0, 1 << min(bits, 63), size=n, dtype=np.uint64)
    keys[: n // 3] = keys[n // 3: 2 * (n // 3)]          # duplicates: stability shows in the values
    return keys, np.arange(n, dtype=np.uint32)


def test_no_alloc_sort_matches_the_allocating_path_twice_in_a_row(ctx):
    import torch
    import paper_2606_23031_b200 as dvx
    cases = [(dvx.SORT_NO_ALLOC_MAX_PAIRS, 42, 1), (100003, 33, 2)]   # 6 passes at the maximum size, then 5 passes on fewer pairs
    dev = []
    for n, bits, seed in cases:
        keys, vals = _pairs(n, bits, seed)
        k_ref = torch.from_numpy(keys.view(np.int64)).cuda()
        v_ref = torch.from_numpy(vals.view(np.int32)).cuda()
        ctx.check(ctx.lib.dvx_sort_pairs(ctx.h, k_ref.data_ptr(), v_ref.data_ptr(), n, bits))   # the existing path
        dev.append((keys, vals, k_ref, v_ref, torch.from_numpy(keys.view(np.int64)).cuda(), torch.from_numpy(vals.view(np.int32)).cuda()))
    torch.cuda.synchronize()
    st = torch.cuda.current_stream().cuda_stream
    # first call (also loads whatever the driver loads lazily), then the second right behind it on the same stream
    dvx.sort_pairs_no_alloc(dev[0][4], dev[0][5], cases[0][1], device=0, stream_ptr=st)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    dvx.sort_pairs_no_alloc(dev[1][4], dev[1][5], cases[1][1], device=0, stream_ptr=st)
    dvx.sort_pairs_no_alloc(dev[0][4], dev[0][5], cases[0][1], device=0, stream_ptr=st)   # sorted input again: still the same result
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the no-alloc entry point changed the device's free memory"
    for (n, bits, _), (keys, vals, k_ref, v_ref, k, v) in zip(cases, dev):
        assert torch.equal(k, k_ref) and torch.equal(v, v_ref), "n = %d, %d bits" % (n, bits)
        order = np.argsort(keys & np.uint64((1 << bits) - 1), kind="stable")       # and both are the stable sort
        assert np.array_equal(k.cpu().numpy().view(np.uint64), keys[order])
        assert np.array_equal(v.cpu().numpy().view(np.uint32), vals[order])


def test_no_alloc_sort_rejects_what_does_not_fit():
    import torch
    import paper_2606_23031_b200 as dvx
    n = dvx.SORT_NO_ALLOC_MAX_PAIRS + 1
    k = torch.zeros(n, dtype=torch.int64, device="cuda")
    v = torch.zeros(n, dtype=torch.int32, device="cuda")
    with pytest.raises(dvx.DvxError) as e:
        dvx.sort_pairs_no_alloc(k, v, 32)
    assert e.value.status == -1 and "DVX_SORT_NO_ALLOC_MAX_PAIRS" in str(e.value)
    with pytest.raises(dvx.DvxError):
        dvx.sort_pairs_no_alloc(k[:8], v[:8], 0)
    dvx.sort_pairs_no_alloc(k[:0], v[:0], 32)     # nothing to do
