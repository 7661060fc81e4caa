"""Parity of mori_eviction_order (CUDA, through the C ABI) with the typed-eviction oracle
(P:L212-221): the victim sequence must be identical page for page, in both tiers."""
import numpy as np
import pytest
import torch

import oracle
from test_oracle_eviction_pins import rand_eviction_case, _gold

pytestmark = pytest.mark.gpu
PAGES = 140000


@pytest.fixture(scope="module", params=["cluster", "multi_kernel"])
def ctx(mori, request):
    """Two sorts behind one entry point: pools of up to 131 072 pages take ONE launch (a cluster of
    8 CTAs), larger ones the general multi-kernel radix sort; MORI_EVICT_MULTI=1 forces the latter
    at every size so that both are checked at every size."""
    import os
    # 32-byte pages: a pool and an arena with many pages cost nothing
    pool = torch.zeros(PAGES * 32, dtype=torch.uint8, device="cuda")
    arena = torch.zeros(PAGES * 32, dtype=torch.uint8).pin_memory()
    if request.param == "multi_kernel":
        os.environ["MORI_EVICT_MULTI"] = "1"
    try:
        m = mori.Mori(1, 1, 8, 1, pool, arena)
    finally:
        os.environ.pop("MORI_EVICT_MULTI", None)
    yield m
    m.close()


def gpu_order(m, which, owner, ptier, last):
    n = len(owner)
    d = "cuda"
    t_o = torch.from_numpy(np.ascontiguousarray(owner, dtype=np.int32)).to(d)
    t_t = torch.from_numpy(np.ascontiguousarray(ptier, dtype=np.uint8)).to(d)
    t_l = torch.from_numpy(np.ascontiguousarray(last, dtype=np.uint32).view(np.int32)).to(d)
    vic = torch.full((max(n, 1),), -7, dtype=torch.int32, device=d)
    nres = torch.full((1,), -7, dtype=torch.int32, device=d)
    m.mori_eviction_order(which, t_o, t_t, t_l, vic, nres)
    torch.cuda.synchronize()
    k = int(nres.item())
    all_pages = vic.cpu().numpy()[:n]
    assert sorted(all_pages.tolist()) == list(range(n))           # a permutation of every page
    return all_pages[:k]


def test_hand_worked_example(ctx, mori):
    g = _gold()
    for which, name in ((mori.TIER_GPU, "gpu"), (mori.TIER_CPU, "cpu")):
        assert gpu_order(ctx, which, g["owner"], g["program_tier"], g["last_access"]).tolist() == g[name].tolist()


@pytest.mark.parametrize("n_pages", [0, 1, 31, 32, 33, 1023, 1024, 1025, 5000, 8191, 8193, 16385, 40960, 65536, 65537, 131072, 131073, PAGES])
def test_random_pools_identical_sequence(ctx, mori, n_pages):
    rng = np.random.default_rng(900 + n_pages)
    for rep in range(3):
        owner, ptier, last = rand_eviction_case(rng, n_pages, int(rng.integers(1, 4097)))
        for which in (mori.TIER_GPU, mori.TIER_CPU):
            got = gpu_order(ctx, which, owner, ptier, last)
            assert np.array_equal(got, oracle.eviction_order(which, owner, ptier, last)), (n_pages, rep, which)


def test_all_free_and_all_one_type(ctx, mori):
    n = 3000
    assert gpu_order(ctx, 0, np.full(n, -1), np.zeros(4, np.uint8), np.zeros(n)).size == 0
    last = np.random.default_rng(1).integers(0, 50, n)
    got = gpu_order(ctx, 1, np.zeros(n, np.int32), np.array([1], np.uint8), last)    # plain LRU, ties by page
    assert np.array_equal(got, np.lexsort((np.arange(n), last)))


def test_argument_errors(ctx, mori):
    z = torch.zeros(8, dtype=torch.int32, device="cuda")
    zt = torch.zeros(8, dtype=torch.uint8, device="cuda")
    with pytest.raises(mori.MoriError):
        ctx.mori_eviction_order(2, z, zt, z, z, z)                   # Waiting is not a pool
    big = torch.zeros(PAGES + 1, dtype=torch.int32, device="cuda")
    with pytest.raises(mori.MoriError):
        ctx.mori_eviction_order(0, big, zt, big, big, z)             # more pages than the pool has
