"""Boundary behaviour of libmori (include/mori.h) that the parity tests do not reach: several live
contexts, the meaning of tickets on every path, MORI_DEBUG validation, stream-ordering calls."""
import os

import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu


def _ctx(mori, L, H, D, T, P, S, path=0, kernel=0, staging=0, seed=1):
    chunk = 2 * H * T * D * 2
    g = torch.Generator(device="cpu").manual_seed(seed)
    pool_h = torch.randint(0, 256, (L * P * chunk,), dtype=torch.uint8, generator=g)
    arena = torch.randint(0, 256, (S * L * chunk,), dtype=torch.uint8, generator=g).pin_memory()
    pool = pool_h.cuda()
    m = mori.Mori(L, H, D, T, pool, arena, path_demote=path, path_promote=path, copy_kernel=kernel,
                  staging_bytes=staging)
    return m, pool, arena, pool_h.numpy().copy(), arena.numpy().copy(), chunk


def test_two_live_contexts_with_different_rings_used_alternately(mori):
    """The bulk-copy kernel's dynamic shared memory limit is a per-function, process-wide
    attribute: a context with small chunks (deep ring of small stages, ~100 KiB) created after one
    with 64 KiB chunks (3 x 64 KiB stages, ~192 KiB) must not lower it under the first."""
    a = _ctx(mori, 3, 8, 128, 16, 200, 200, path=2, kernel=2, seed=1)       # 64 KiB chunks
    b = _ctx(mori, 2, 2, 32, 8, 300, 300, path=2, kernel=2, seed=2)         # 2 KiB chunks, created second
    rng = np.random.default_rng(0)
    for rep in range(3):
        for (m, pool, arena, pool_m, arena_m, chunk), (L, P, S) in ((a, (3, 200, 200)), (b, (2, 300, 300))):
            g = rng.permutation(P)[:150].astype(np.int32)
            h = rng.permutation(S)[:150].astype(np.int32)
            m.mori_demote(g, h)
            m.mori_sync(mori.BOTH)
            oracle.demote(L, chunk, pool_m, arena_m, g, h)
            assert np.array_equal(arena.numpy(), arena_m), rep
            g2 = rng.permutation(P)[:150].astype(np.int32)
            m.mori_promote(h, g2)
            m.mori_sync(mori.BOTH)
            oracle.promote(L, chunk, pool_m, arena_m, h, g2)
            assert np.array_equal(pool.cpu().numpy(), pool_m), rep
    a[0].close()
    b[0].close()


@pytest.mark.parametrize("path", [0, 1, 2, 3])
@pytest.mark.parametrize("slot_runs", ["one_run", "scattered"])
def test_ticket_orders_arena_reads_after_the_demote_on_every_path(mori, path, slot_runs):
    """demote(slots) then promote(slots, slots_after_demote = its ticket) with NO join in between:
    the promotion must read what the demotion wrote, whichever path each call takes (AUTO picks
    STAGED for one long run of slots and ZEROCOPY for scattered ones)."""
    L, H, D, T, P, S = 4, 8, 128, 16, 3000, 3000               # 256 KiB pages
    m, pool, arena, pool_m, arena_m, chunk = _ctx(mori, L, H, D, T, P, S, path=path, kernel=2, seed=3)
    rng = np.random.default_rng(7)
    k = 1400                                                    # 350 MiB: the demotion takes milliseconds
    for rep in range(2):
        g = rng.permutation(P)[:k].astype(np.int32)
        h = (np.arange(k) + 100 * rep if slot_runs == "one_run" else rng.permutation(S // 2)[:k] * 2).astype(np.int32)
        g2 = np.setdiff1d(np.arange(P, dtype=np.int32), g)[:k]  # fresh pages: the pool ticket is not what is tested
        t = m.mori_demote(g, h)
        m.mori_promote(h, g2, slots_after_demote=t)
        m.mori_sync(mori.BOTH)
        oracle.demote(L, chunk, pool_m, arena_m, g, h)
        oracle.promote(L, chunk, pool_m, arena_m, h, g2)
        assert np.array_equal(arena.numpy(), arena_m), (rep, "arena")
        assert np.array_equal(pool.cpu().numpy(), pool_m), (rep, "pool: the promotion read stale arena bytes")
    m.close()


@pytest.mark.parametrize("path", [0, 1, 2])
def test_ticket_orders_pool_writes_after_the_demote_that_vacates_the_pages(mori, path):
    """promote into the very pages a demotion of the same epoch is reading, no join: the demotion
    must have read them first (pages_after_demote)."""
    L, H, D, T, P, S = 4, 8, 128, 16, 1500, 3000
    m, pool, arena, pool_m, arena_m, chunk = _ctx(mori, L, H, D, T, P, S, path=path, kernel=2, seed=4)
    rng = np.random.default_rng(8)
    g = rng.permutation(P)[:1400].astype(np.int32)
    h_out = np.arange(1400, dtype=np.int32)
    h_in = (1500 + np.arange(1400)).astype(np.int32)           # slots that already hold (random) bytes
    t = m.mori_demote(g, h_out)
    m.mori_promote(h_in, g[::-1].copy(), pages_after_demote=t)
    m.mori_sync(mori.BOTH)
    oracle.demote(L, chunk, pool_m, arena_m, g, h_out)
    oracle.promote(L, chunk, pool_m, arena_m, h_in, g[::-1].copy())
    assert np.array_equal(arena.numpy(), arena_m), "the demotion read pages the promotion had already overwritten"
    assert np.array_equal(pool.cpu().numpy(), pool_m)
    m.close()


def test_small_calls_take_one_launch_and_are_byte_exact(mori):
    """AUTO: a call of a few pages (cfg 1: KiBs) is ONE kernel launch with the ids in its
    parameters -- no index upload, no staging, no DMA."""
    L, H, D, T, P, S = 2, 2, 64, 16, 64, 256                    # cfg-1 geometry: 16 KiB pages
    m, pool, arena, pool_m, arena_m, chunk = _ctx(mori, L, H, D, T, P, S, path=0, kernel=0, seed=5)
    rng = np.random.default_rng(9)
    for k in (1, 2, 25, 64):
        g = rng.permutation(P)[:k].astype(np.int32)
        h = rng.permutation(S)[:k].astype(np.int32)
        l0 = m.mori_launch_count()
        t = m.mori_demote(g, h)
        assert m.mori_launch_count() - l0 == 1
        g2 = rng.permutation(P)[:k].astype(np.int32)
        l0 = m.mori_launch_count()
        m.mori_promote(h, g2, pages_after_demote=t, slots_after_demote=t)
        assert m.mori_launch_count() - l0 == 1
        m.mori_sync(mori.BOTH)
        oracle.demote(L, chunk, pool_m, arena_m, g, h)
        oracle.promote(L, chunk, pool_m, arena_m, h, g2)
        assert np.array_equal(arena.numpy(), arena_m), k
        assert np.array_equal(pool.cpu().numpy(), pool_m), k
    m.close()


def test_mori_debug_finds_duplicate_destinations(mori):
    os.environ["MORI_DEBUG"] = "1"
    try:
        m, pool, arena, pool_m, arena_m, chunk = _ctx(mori, 2, 2, 64, 16, 64, 64, path=2, kernel=2, seed=6)
    finally:
        del os.environ["MORI_DEBUG"]
    ok = np.arange(8, dtype=np.int32)
    dup = np.array([0, 1, 2, 3, 4, 5, 6, 3], np.int32)
    with pytest.raises(mori.MoriError) as e:
        m.mori_demote(ok, dup)                                  # two pages into one slot
    assert e.value.code == mori.ERR_INVALID_ARG and "duplicate" in str(e.value)
    with pytest.raises(mori.MoriError) as e:
        m.mori_promote(ok, dup)                                 # two slots into one page
    assert e.value.code == mori.ERR_INVALID_ARG
    m.mori_demote(dup, ok)                                      # duplicate SOURCES are fine
    m.mori_promote(dup, ok)
    m.mori_demote(ok, ok)                                       # and the scratch bitmap is clean again
    m.mori_sync(mori.BOTH)
    stg = torch.zeros(8 * 2 * chunk, dtype=torch.uint8, device="cuda")
    with pytest.raises(mori.MoriError) as e:
        m.mori_scatter_pages(torch.from_numpy(dup).cuda(), stg)
    assert e.value.code == mori.ERR_INVALID_ARG
    with pytest.raises(mori.MoriError):
        m.mori_gather_pages(torch.from_numpy(np.array([0, 64], np.int32)).cuda(), stg)   # out of range
    m.mori_gather_pages(torch.from_numpy(dup).cuda(), stg)      # duplicate sources are fine
    m.mori_scatter_pages(torch.from_numpy(ok).cuda(), stg)
    torch.cuda.synchronize()
    m.close()
    # release contexts do not pay for the check and do not reject the table
    m2, *_ = _ctx(mori, 2, 2, 64, 16, 64, 64, path=2, kernel=2, seed=6)
    m2.mori_demote(ok, dup)
    m2.mori_sync(mori.BOTH)
    m2.close()


def test_stream_ordering_calls_check_their_arguments(mori):
    m, *_ = _ctx(mori, 2, 2, 64, 16, 16, 16, seed=7)
    s = torch.cuda.Stream()
    for which in (0, 4, -1):
        assert m._lib.mori_after_stream(m._h, which, s.cuda_stream) == mori.ERR_INVALID_ARG
        assert m._lib.mori_stream_wait(m._h, s.cuda_stream, which) == mori.ERR_INVALID_ARG
    assert m._lib.mori_after_stream(None, 3, s.cuda_stream) == mori.ERR_INVALID_ARG
    assert m._lib.mori_stream_wait(None, s.cuda_stream, 3) == mori.ERR_INVALID_ARG
    m.mori_after_stream(mori.BOTH, s)
    m.mori_stream_wait(s, mori.BOTH)
    s.synchronize()
    m.close()


def test_eviction_order_alternating_tiers_keeps_both_graphs(mori):
    """The GPU-tier and CPU-tier orders called alternately (what an engine does every tick) must
    each stay correct; the library keeps one captured graph per tier."""
    P, S, n = 3000, 5000, 64
    pool = torch.zeros(P * 32, dtype=torch.uint8, device="cuda")
    arena = torch.zeros(S * 32, dtype=torch.uint8).pin_memory()
    m = mori.Mori(1, 1, 8, 1, pool, arena)
    rng = np.random.default_rng(5)
    dev = lambda x: torch.from_numpy(x).cuda()
    tabs = {}
    for which, N in ((mori.TIER_GPU, P), (mori.TIER_CPU, S)):
        owner = rng.integers(-1, n, N).astype(np.int32)
        last = rng.integers(0, 500, N).astype(np.uint32)
        tabs[which] = (owner, last, dev(owner), dev(last.view(np.int32)),
                       torch.empty(N, dtype=torch.int32, device="cuda"), torch.empty(1, dtype=torch.int32, device="cuda"))
    ptier = rng.integers(0, 3, n).astype(np.uint8)
    d_ptier = dev(ptier)
    for rep in range(4):
        for which in (mori.TIER_GPU, mori.TIER_CPU):
            owner, last, d_o, d_l, vic, nres = tabs[which]
            m.mori_eviction_order(which, d_o, d_ptier, d_l, vic, nres)
            torch.cuda.synchronize()
            want = oracle.eviction_order(0 if which == mori.TIER_GPU else 1, owner, ptier, last)
            assert np.array_equal(vic.cpu().numpy()[:int(nres.item())], want), (rep, which)
    m.close()


def test_profile_timeline_and_launch_floor(mori):
    """mori_profile(ctx, 2) keeps every kernel and every staging segment's DMAs of a call as
    [start, end) on one clock; mori_noop is one (empty) launch."""
    L, H, D, T, P, S = 2, 8, 128, 16, 256, 256                  # 128 KiB pages
    chunk = 2 * H * T * D * 2
    m, pool, arena, pool_m, arena_m, _ = _ctx(mori, L, H, D, T, P, S, path=2, kernel=2, staging=40 * L * chunk, seed=8)
    g = np.arange(100, dtype=np.int32)
    h = np.arange(100, dtype=np.int32)
    m.mori_profile(2)
    m.mori_demote(g, h)
    m.mori_promote(h, (g + 120).astype(np.int32))
    m.mori_sync(mori.BOTH)
    for which in (mori.DEMOTE, mori.PROMOTE):
        rows = m.mori_profile_timeline(which)
        kern = [r for r in rows if r[0] == 0]
        dma = [r for r in rows if r[0] == 1]
        assert len(kern) == len(dma) == 3                        # segments of 40, 40, 20 pages
        assert sum(r[3] for r in kern) == sum(r[3] for r in dma) == 100 * L * chunk
        assert all(0 <= r[1] < r[2] for r in rows)
        for k, d in zip(sorted(kern, key=lambda r: r[1]), sorted(dma, key=lambda r: r[1])):
            if which == mori.DEMOTE:
                assert k[2] <= d[1] + 1e-3                       # a segment's DMA follows its gather
            else:
                assert d[2] <= k[1] + 1e-3                       # a segment's scatter follows its DMA
    ms, launches, nbytes = m.mori_profile_read(mori.DEMOTE)
    assert launches == 3 and nbytes == 100 * L * chunk           # kernels only, as with mori_profile(1)
    m.mori_profile(False)
    l0 = m.mori_launch_count()
    m.mori_noop()
    torch.cuda.synchronize()
    assert m.mori_launch_count() - l0 == 1
    oracle.demote(L, chunk, pool_m, arena_m, g, h)
    oracle.promote(L, chunk, pool_m, arena_m, h, (g + 120).astype(np.int32))
    assert np.array_equal(arena.numpy(), arena_m) and np.array_equal(pool.cpu().numpy(), pool_m)
    m.close()


def test_after_stream_is_lazy_but_still_orders_every_library_stream(mori):
    """mori_after_stream only records an event; a library stream waits on it when it next gets work.
    A side stream sleeps, then rewrites the whole pool and the whole arena.  A small demotion (one
    launch on the kernel stream) and a large STAGED promotion (whose first operations are DMAs on the
    DMA stream) issued right after mori_after_stream must both see the NEW bytes."""
    L, H, D, T, P, S = 2, 8, 128, 16, 700, 700                   # 128 KiB pages
    m, pool, arena, pool_m, arena_m, chunk = _ctx(mori, L, H, D, T, P, S, path=0, kernel=0, seed=11)
    g = torch.Generator(device="cpu").manual_seed(12)
    new_pool = torch.randint(0, 256, (pool.numel(),), dtype=torch.uint8, generator=g)
    new_arena = torch.randint(0, 256, (arena.numel(),), dtype=torch.uint8, generator=g)
    d_new_pool, d_new_arena = new_pool.cuda(), new_arena.cuda()
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    for rep in range(2):                                          # the second round reuses a recycled event
        with torch.cuda.stream(side):
            torch.cuda._sleep(40_000_000)                         # ~20 ms: the library would win any race
            pool.copy_(d_new_pool)
            arena.copy_(d_new_arena, non_blocking=True)
        m.mori_after_stream(mori.BOTH, side)
        g_small = np.array([3, 699, 42, 7], np.int32)
        h_small = np.array([650, 2, 651, 699], np.int32)
        g_big = (100 + np.arange(500)).astype(np.int32)
        h_big = (100 + np.arange(500)).astype(np.int32)            # one run of 62.5 MiB -> STAGED
        l0 = m.mori_launch_count()
        m.mori_demote(g_small, h_small)
        assert m.mori_launch_count() - l0 == 1                     # the one-launch path
        m.mori_promote(h_big, g_big[::-1].copy())
        m.mori_sync(mori.BOTH)
        side.synchronize()
        pool_m, arena_m = new_pool.numpy().copy(), new_arena.numpy().copy()
        oracle.demote(L, chunk, pool_m, arena_m, g_small, h_small)
        oracle.promote(L, chunk, pool_m, arena_m, h_big, g_big[::-1].copy())
        assert np.array_equal(arena.numpy(), arena_m), (rep, "the demotion did not wait for the side stream")
        assert np.array_equal(pool.cpu().numpy(), pool_m), (rep, "the promotion's DMAs did not wait for the side stream")
        # restore different contents for the next round, so that stale data would show
        d_new_pool, d_new_arena = d_new_pool.flip(0).contiguous(), d_new_arena.flip(0).contiguous()
        new_pool, new_arena = new_pool.flip(0).contiguous(), new_arena.flip(0).contiguous()
    # many after_stream calls with no work and no join in between must not grow without bound
    for _ in range(100):
        m.mori_after_stream(mori.BOTH, side)
    m.mori_demote(np.array([1], np.int32), np.array([1], np.int32))
    m.mori_sync(mori.BOTH)
    m.close()
