"""Parity of mori_demote / mori_promote / gather / scatter (CUDA, through the C ABI) with the CPU
oracle's per-page memcpy: byte-exact pools and arenas, every path and both copy kernels."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_00866_b200 import workload as W
from paper_2606_00866_b200.harness import GpuRunner

pytestmark = pytest.mark.gpu

PATHS = [0, 1, 2, 3]       # auto (per call), zerocopy, staged, copyengine
KERNELS = [1, 2]           # ldst, tma


def _mk_ctx(mori, L, H, D, T, P, S, path, kernel, staging=0):
    chunk = 2 * H * T * D * 2
    g = torch.Generator(device="cpu").manual_seed(P * 31 + S)
    pool_h = torch.randint(0, 256, (L * P * chunk,), dtype=torch.uint8, generator=g)
    arena = torch.randint(0, 256, (S * L * chunk,), dtype=torch.uint8, generator=g).pin_memory()
    pool = pool_h.cuda()
    m = mori.Mori(L, H, D, T, pool, arena, path_demote=path, path_promote=path, copy_kernel=kernel,
                  staging_bytes=staging)
    return m, pool, arena, pool_h.numpy().copy(), arena.numpy().copy(), chunk


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape", [(2, 2, 64, 16, 64, 256),        # cfg-1 geometry: 8 KiB chunks
                                   (5, 8, 128, 16, 300, 200),      # 64 KiB chunks
                                   (3, 8, 128, 32, 70, 90),        # 128 KiB chunks
                                   (3, 1, 24, 5, 50, 40)])         # ragged: 960-byte chunks
def test_demote_then_promote_byte_exact(mori, path, kernel, shape):
    L, H, D, T, P, S = shape
    # small staging so that STAGED runs several segments with a ragged last one
    m, pool, arena, pool_m, arena_m, chunk = _mk_ctx(mori, L, H, D, T, P, S, path, kernel,
                                                      staging=7 * L * 2 * H * T * D * 2)
    rng = np.random.default_rng(P)
    k = min(P, S) // 2 + 3
    g = rng.permutation(P)[:k].astype(np.int32)
    h = rng.permutation(S)[:k].astype(np.int32)
    h[: k // 2] = np.sort(h[: k // 2])                       # some consecutive-slot runs
    t = m.mori_demote(g, h)
    assert t > 0
    m.mori_sync(mori.DEMOTE)
    oracle.demote(L, chunk, pool_m, arena_m, g, h)
    assert np.array_equal(arena.numpy(), arena_m), "arena differs after demote"
    assert np.array_equal(pool.cpu().numpy(), pool_m), "pool changed by demote"
    g2 = rng.permutation(P)[:k].astype(np.int32)
    m.mori_promote(h, g2, pages_after_demote=t, slots_after_demote=t)
    m.mori_sync(mori.BOTH)
    oracle.promote(L, chunk, pool_m, arena_m, h, g2)
    assert np.array_equal(pool.cpu().numpy(), pool_m), "pool differs after promote"
    assert np.array_equal(arena.numpy(), arena_m), "arena changed by promote"
    # empty calls are valid no-ops that still issue tickets
    e = np.zeros(0, np.int32)
    assert m.mori_demote(e, e) > t
    assert m.mori_promote(e, e) > 0
    m.mori_sync(mori.BOTH)
    assert np.array_equal(pool.cpu().numpy(), pool_m)
    m.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_gather_scatter_device(mori, kernel):
    L, H, D, T, P = 4, 8, 128, 16, 400
    m, pool, arena, pool_m, arena_m, chunk = _mk_ctx(mori, L, H, D, T, P, 8, 2, kernel)
    rng = np.random.default_rng(3)
    g = rng.permutation(P)[:157].astype(np.int32)
    gd = torch.from_numpy(g).cuda()
    stg = torch.zeros(157 * L * chunk, dtype=torch.uint8, device="cuda")
    m.mori_gather_pages(gd, stg)
    torch.cuda.synchronize()
    want = np.zeros(157 * L * chunk, np.uint8)
    oracle.demote(L, chunk, pool_m, want, g, np.arange(157, dtype=np.int32))
    assert np.array_equal(stg.cpu().numpy(), want)
    g2 = rng.permutation(P)[:157].astype(np.int32)
    m.mori_scatter_pages(torch.from_numpy(g2).cuda(), stg)
    torch.cuda.synchronize()
    oracle.promote(L, chunk, pool_m, want, np.arange(157, dtype=np.int32), g2)
    assert np.array_equal(pool.cpu().numpy(), pool_m)
    m.mori_gather_pages(gd[:0], stg)           # empty
    m.close()


def test_migration_argument_errors(mori):
    m, pool, arena, *_ = _mk_ctx(mori, 2, 2, 64, 16, 16, 8, 2, 2)
    one = np.array([0], np.int32)
    for g, h in [(np.array([16], np.int32), one), (np.array([-1], np.int32), one),
                 (one, np.array([8], np.int32)), (one, np.array([-1], np.int32))]:
        with pytest.raises(mori.MoriError) as e:
            m.mori_demote(g, h)
        assert e.value.code == mori.ERR_INVALID_ARG
        with pytest.raises(mori.MoriError):
            m.mori_promote(h, g)
    with pytest.raises(mori.MoriError):
        m.mori_promote(one, one, pages_after_demote=12345)          # never issued
    with pytest.raises(mori.MoriError):
        m.mori_sync(0)
    m.mori_sync(mori.BOTH)
    m.close()
    # no arena -> STATE error
    m2 = mori.Mori(2, 2, 64, 16, pool)
    with pytest.raises(mori.MoriError) as e:
        m2.mori_demote(one, one)
    assert e.value.code == mori.ERR_STATE
    m2.close()


def test_device_fill_matches_numpy_generator(mori):
    cfg = W.get_config(1)
    r = GpuRunner(cfg, 866)
    pages = np.array([5, 0, 63, 17], np.int32)
    r.fill([(42, 3, pages)])
    pv = r.pool.cpu().numpy().reshape(cfg.shape.n_layers, cfg.gpu_pool_pages, cfg.shape.chunk_bytes)
    for j, g in enumerate(pages):
        assert np.array_equal(pv[:, g], W.page_content(866, 42, 3 + j, cfg.shape))
    assert r.check([(42, 3, pages)]) == 0
    assert r.check([(42, 4, pages)]) > 0
    r.close()


def _epochs_with_mirror(mori, cfg, seed, epochs, path, kernel, sticky=False):
    """Whole epochs: GPU placement must equal the oracle's; the CUDA movers and the oracle's
    memcpy movers get identical tables; both pools are compared byte for byte every epoch."""
    sh = cfg.shape
    sim = W.Sim(cfg, seed)
    r = GpuRunner(cfg, seed, path_demote=path, path_promote=path, copy_kernel=kernel,
                  staging_bytes=max(sh.page_bytes * 3, 1 << 20))
    pool_m = np.zeros(sh.n_layers * cfg.gpu_pool_pages * sh.chunk_bytes, np.uint8)
    arena_m = np.zeros(cfg.cpu_pool_pages * sh.page_bytes, np.uint8)
    r.arena.zero_()
    moved = 0
    for e in range(epochs):
        plan = sim.begin_epoch()
        if sticky:
            want = oracle.sticky_rebalance(plan.iota, plan.kv_pages, plan.prev_tier, plan.flags,
                                           cfg.cap_gpu_pages, cfg.cap_cpu_pages)
            got = r.place_sticky(plan.iota, plan.kv_pages, plan.prev_tier, plan.flags)
            keys = ("tier", "lazy", "used")
        else:
            want = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
            got = r.place(plan.iota, plan.kv_pages, plan.prev_tier)
            keys = ("order", "tier", "bounds", "used")
        for k in keys:
            assert np.array_equal(got[k], want[k]), (cfg.name, e, k)
        for k in range(5):
            assert np.array_equal(got["lists"][k], want["lists"][k]), (cfg.name, e, k)
        sim.apply_placement(got["tier"], got["lists"])
        r.execute(plan)
        for op in plan.ops:
            if op[0] == "demote":
                oracle.demote(sh.n_layers, sh.chunk_bytes, pool_m, arena_m, op[3], op[4])
            elif op[0] == "promote":
                oracle.promote(sh.n_layers, sh.chunk_bytes, pool_m, arena_m, op[3], op[4])
        sim.end_epoch()
        r.fill(plan.fills)
        pv = pool_m.reshape(sh.n_layers, cfg.gpu_pool_pages, sh.chunk_bytes)
        for uid, first, pages in plan.fills:
            for j, g in enumerate(pages):
                pv[:, g] = W.page_content(seed, uid, first + j, sh)
        assert np.array_equal(r.pool.cpu().numpy(), pool_m), (cfg.name, e, "pool")
        assert np.array_equal(r.arena.numpy(), arena_m), (cfg.name, e, "arena")
        moved += plan.demote_pages + plan.promote_pages
    gtri, htri = r.resident(sim)
    assert r.check(gtri) == 0 and r.check(htri, arena=True) == 0
    r.close()
    return moved


@pytest.mark.parametrize("path", PATHS)
def test_cfg1_epochs_full_mirror(mori, path):
    for seed in (866, 867, 868):
        _epochs_with_mirror(mori, W.get_config(1), seed, 20, path, 2)


# (zero-copy path, LD/ST kernel) and (staged path, bulk-copy kernel); cfg 3 and 4 run the first pair
# in the sweep test below (AUTO) and in the mover tests above, which keeps the suite inside its budget
@pytest.mark.parametrize("idx,scale,epochs,path,kernel", [(2, 128, 20, 1, 1), (2, 128, 20, 2, 2), (3, 128, 12, 2, 2),
                                                          (4, 128, 10, 2, 2), (5, 128, 10, 1, 1), (5, 128, 10, 2, 2)])
def test_scaled_twins_epochs_full_mirror(mori, idx, scale, epochs, path, kernel):
    moved = _epochs_with_mirror(mori, W.get_config(idx, scale), 866, epochs, path, kernel)
    assert moved > 0


@pytest.mark.parametrize("f_busy", [0.25, 0.5, 0.75])
def test_cfg3_busy_idle_sweep_epochs_full_mirror(mori, f_busy):
    """BASELINE.json configs[2]: the busy:idle ratio swept 1:3, 1:1, 3:1.  Scaled twin with byte
    mirrors of both pools, AUTO paths (the library picks per call), 12 epochs each."""
    moved = _epochs_with_mirror(mori, W.get_config(3, 128, f_busy), 866, 12, 0, 0)
    assert moved > 0


def test_merged_and_per_program_calls_move_the_same_bytes(mori):
    """The harness issues an epoch's demotions as one flat call (a move is a list of pages); one call
    per program must leave both pools in the same state."""
    cfg = W.get_config(2, 128)
    sh = cfg.shape
    states = []
    for merge in (True, False):
        sim = W.Sim(cfg, 867)
        r = GpuRunner(cfg, 867, staging_bytes=sh.page_bytes * 5)
        r.arena.zero_()
        for e in range(12):
            plan = sim.begin_epoch()
            got = r.place(plan.iota, plan.kv_pages, plan.prev_tier)
            sim.apply_placement(got["tier"], got["lists"])
            r.execute(plan, merge=merge)
            sim.end_epoch()
            r.fill(plan.fills)
        states.append((r.pool.cpu().numpy().copy(), r.arena.numpy().copy()))
        r.close()
    assert np.array_equal(states[0][0], states[1][0]) and np.array_equal(states[0][1], states[1][1])


@pytest.mark.parametrize("idx,scale,epochs", [(2, 128, 30)])
def test_sticky_policy_epochs_full_mirror(mori, idx, scale, epochs):
    """NEXT-1 end to end: placement from mori_sticky_rebalance (== the section-4.3.1 oracle every
    epoch), bytes moved by mori_demote / mori_promote, both pools mirrored byte for byte."""
    moved = _epochs_with_mirror(mori, W.get_config(idx, scale), 866, epochs, 0, 2, sticky=True)
    assert moved > 0


@pytest.mark.parametrize("path", [1, 2])
def test_many_calls_without_a_join_wrap_the_index_ring(mori, path):
    """The library stages page/slot ids in a pinned ring (64 Ki entries at least); 700 calls of 60
    pages with no mori_sync in between overflow it, which must drain the streams and carry on."""
    L, H, D, T, P, S = 1, 1, 8, 1, 4096, 4096            # 32-byte pages
    m, pool, arena, pool_m, arena_m, chunk = _mk_ctx(mori, L, H, D, T, P, S, path, 2, staging=64 * 32)
    rng = np.random.default_rng(11)
    for call in range(700):
        g = rng.integers(0, P, 60).astype(np.int32)
        h = rng.permutation(S)[:60].astype(np.int32)
        m.mori_demote(g, h)
        oracle.demote(L, chunk, pool_m, arena_m, g, h)       # later calls overwrite earlier slots: order matters
    m.mori_sync(mori.BOTH)
    assert np.array_equal(arena.numpy(), arena_m)
    for call in range(700):
        h = rng.integers(0, S, 60).astype(np.int32)
        g = rng.permutation(P)[:60].astype(np.int32)
        m.mori_promote(h, g)
        oracle.promote(L, chunk, pool_m, arena_m, h, g)
    m.mori_sync(mori.BOTH)
    assert np.array_equal(pool.cpu().numpy(), pool_m)
    m.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_device_resident_arena_is_a_third_tier(mori, kernel):
    """The arena may be device memory (a peer GPU's HBM over NVLink in production; a second
    buffer of the same GPU here): demote / promote byte-exact against the oracle, one kernel each."""
    L, H, D, T, P, S = 4, 8, 128, 16, 300, 260
    chunk = 2 * H * T * D * 2
    g0 = torch.Generator(device="cpu").manual_seed(5)
    pool_h = torch.randint(0, 256, (L * P * chunk,), dtype=torch.uint8, generator=g0)
    arena_h = torch.randint(0, 256, (S * L * chunk,), dtype=torch.uint8, generator=g0)
    pool, arena = pool_h.cuda(), arena_h.cuda()
    m = mori.Mori(L, H, D, T, pool, arena, copy_kernel=kernel)
    assert m.path_demote == mori.PATH_ZEROCOPY and m.path_promote == mori.PATH_ZEROCOPY
    pool_m, arena_m = pool_h.numpy().copy(), arena_h.numpy().copy()
    rng = np.random.default_rng(2)
    g = rng.permutation(P)[:200].astype(np.int32); h = rng.permutation(S)[:200].astype(np.int32)
    l0 = m.mori_launch_count()
    t = m.mori_demote(g, h)
    m.mori_sync(mori.BOTH)
    assert m.mori_launch_count() - l0 == 2                    # index upload + one copy kernel
    oracle.demote(L, chunk, pool_m, arena_m, g, h)
    assert np.array_equal(arena.cpu().numpy(), arena_m) and np.array_equal(pool.cpu().numpy(), pool_m)
    g2 = rng.permutation(P)[:200].astype(np.int32)
    m.mori_promote(h, g2, pages_after_demote=t, slots_after_demote=t)
    m.mori_sync(mori.BOTH)
    oracle.promote(L, chunk, pool_m, arena_m, h, g2)
    assert np.array_equal(pool.cpu().numpy(), pool_m) and np.array_equal(arena.cpu().numpy(), arena_m)
    m.close()


def test_auto_keeps_issue_order_when_consecutive_calls_take_different_paths(mori):
    """AUTO picks STAGED for a long run of slots and ZEROCOPY for scattered ones; two demotes in a
    row that write the same slots must still land in issue order (the second one wins)."""
    L, H, D, T, P, S = 4, 8, 128, 16, 2048, 2048               # 256 KiB pages
    m, pool, arena, pool_m, arena_m, chunk = _mk_ctx(mori, L, H, D, T, P, S, 0, 2)
    rng = np.random.default_rng(4)
    for rep in range(3):
        g_a = rng.permutation(P)[:1500].astype(np.int32)
        h_a = np.arange(1500, dtype=np.int32)                  # one run of 375 MiB -> STAGED (a long DMA)
        g_b = rng.permutation(P)[:300].astype(np.int32)
        h_b = (rng.permutation(750)[:300] * 2).astype(np.int32)   # isolated slots inside that run -> ZEROCOPY
        m.mori_demote(g_a, h_a)
        m.mori_demote(g_b, h_b)
        m.mori_sync(mori.BOTH)
        oracle.demote(L, chunk, pool_m, arena_m, g_a, h_a)
        oracle.demote(L, chunk, pool_m, arena_m, g_b, h_b)
        assert np.array_equal(arena.numpy(), arena_m), rep
    m.close()


def test_profile_counts_the_gather_launches_of_a_staged_call(mori):
    L, H, D, T, P, S = 2, 8, 128, 16, 64, 64
    chunk = 2 * H * T * D * 2
    m, pool, arena, pool_m, arena_m, _ = _mk_ctx(mori, L, H, D, T, P, S, 2, 2, staging=10 * L * chunk)
    g = np.arange(25, dtype=np.int32); h = np.arange(25, dtype=np.int32)
    m.mori_profile(True)
    l0 = m.mori_launch_count()
    m.mori_demote(g, h)
    m.mori_sync(mori.BOTH)
    ms, launches, nbytes = m.mori_profile_read(mori.DEMOTE)
    assert launches == 3 and nbytes == 25 * L * chunk and ms > 0          # segments of 10, 10, 5 pages
    assert m.mori_launch_count() - l0 == 4                                # + the index upload
    assert m.mori_profile_read(mori.DEMOTE) == (0.0, 0, 0)                # read clears
    assert m.mori_profile_read(mori.PROMOTE) == (0.0, 0, 0)
    m.mori_profile(False)
    m.mori_demote(g, h)
    m.mori_sync(mori.BOTH)
    assert m.mori_profile_read(mori.DEMOTE) == (0.0, 0, 0)
    m.close()
