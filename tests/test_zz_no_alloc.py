"""mori_eviction_order_noalloc -- the entry point for callers that cannot call cudaMalloc (code under
CUDA graph capture, tight serving loops): its sort scratch is a 1 MiB file-scope static device array.
Its victim sequence must equal the existing path's (mori_eviction_order, which allocates its scratch)
page for page -- integer output, so bit-exact like every other eviction test -- on two calls in a row
that share the scratch, and the oracle's.  Collected last on purpose (the suite runs with pytest -x);
passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu


def _case(rng, n_pages, n_programs, hi):
    owner = rng.integers(-1, n_programs, n_pages).astype(np.int32)
    ptier = rng.integers(0, 3, n_programs).astype(np.uint8)
    last = rng.integers(0, hi, n_pages, dtype=np.uint64).astype(np.uint32)
    return owner, ptier, last


def _dev(owner, ptier, last):
    d = "cuda"
    return (torch.from_numpy(owner).to(d), torch.from_numpy(ptier).to(d),
            torch.from_numpy(last.view(np.int32)).to(d))


def test_no_alloc_entry_point_equals_the_existing_path_on_two_calls_in_a_row(mori):
    n_max = mori.Mori.NOALLOC_MAX_PAGES
    pool = torch.zeros(n_max * 32, dtype=torch.uint8, device="cuda")          # 32-byte pages
    arena = torch.zeros(n_max * 32, dtype=torch.uint8).pin_memory()
    m = mori.Mori(1, 1, 8, 1, pool, arena)
    rng = np.random.default_rng(424242)
    # two calls in a row on one stream, the second SMALLER and on different data: stale contents of
    # the shared scratch from the first call would show up in it; then the maximum size, both tiers
    calls = [(mori.TIER_GPU, 40960, 300, 2 ** 32), (mori.TIER_CPU, 5000, 64, 200),
             (mori.TIER_GPU, n_max, 4096, 1000), (mori.TIER_CPU, n_max, 64, 2 ** 32), (mori.TIER_GPU, 1, 1, 5)]
    outs = []
    for which, n, n_prog, hi in calls:                                     # enqueue everything, no sync in between
        owner, ptier, last = _case(rng, n, n_prog, hi)
        d_o, d_t, d_l = _dev(owner, ptier, last)
        vic = torch.full((n,), -7, dtype=torch.int32, device="cuda")
        nres = torch.full((1,), -7, dtype=torch.int32, device="cuda")
        mori.Mori.mori_eviction_order_noalloc(which, d_o, d_t, d_l, vic, nres)
        outs.append((which, owner, ptier, last, d_o, d_t, d_l, vic, nres))
    torch.cuda.synchronize()
    for which, owner, ptier, last, d_o, d_t, d_l, vic, nres in outs:
        n = owner.size
        ref_vic = torch.full((n,), -9, dtype=torch.int32, device="cuda")
        ref_n = torch.full((1,), -9, dtype=torch.int32, device="cuda")
        m.mori_eviction_order(which, d_o, d_t, d_l, ref_vic, ref_n)           # the existing (allocating) path
        torch.cuda.synchronize()
        k = int(ref_n.item())
        assert int(nres.item()) == k, (which, n)
        got = vic.cpu().numpy()
        assert np.array_equal(got[:k], ref_vic.cpu().numpy()[:k]), (which, n, "differs from mori_eviction_order")
        assert sorted(got.tolist()) == list(range(n))                          # a permutation of every page
        want = oracle.eviction_order(0 if which == mori.TIER_GPU else 1, owner, ptier, last)
        assert np.array_equal(got[:k], want), (which, n, "differs from the oracle")
    m.close()


def test_no_alloc_entry_point_rejects_sizes_beyond_its_static_scratch(mori):
    n = mori.Mori.NOALLOC_MAX_PAGES + 1
    z = torch.zeros(n, dtype=torch.int32, device="cuda")
    t = torch.zeros(4, dtype=torch.uint8, device="cuda")
    nres = torch.full((1,), 5, dtype=torch.int32, device="cuda")
    with pytest.raises(mori.MoriError) as e:
        mori.Mori.mori_eviction_order_noalloc(mori.TIER_GPU, z, t, z, z, nres)
    assert e.value.code == mori.ERR_CAPACITY and "MORI_NOALLOC_MAX_PAGES" in str(e.value)
    with pytest.raises(mori.MoriError) as e:
        mori.Mori.mori_eviction_order_noalloc(2, z[:8], t, z[:8], z[:8], nres)   # Waiting is not a pool
    assert e.value.code == mori.ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert int(nres.item()) == 5                                               # nothing was enqueued
    mori.Mori.mori_eviction_order_noalloc(mori.TIER_CPU, z[:0], t, z[:0], z[:0], nres)   # empty pool: a valid no-op
    torch.cuda.synchronize()
    assert int(nres.item()) == 0
