"""Pins of the T-tier partition oracle (NEXT-4(ii)): T = 2 is the already pinned
rank/partition, a cumsum/searchsorted restatement, a brute force over all 4^n maps for T = 3, and
a hand-checkable case.  CPU only."""
import itertools

import numpy as np
import pytest

import oracle
from oracle import oracle_np
from test_oracle_pins import _rand_case


def test_hand_checkable_three_tiers():
    # ranking by iota: p3(.1) p0(.2) p4(.3) p1(.6) p2(.9); sizes in that order 2 3 4 1 5
    r = oracle.rank_partition_tiers([0.2, 0.6, 0.9, 0.1, 0.3], [3, 1, 5, 2, 4], [5, 4, 1])
    assert r["order"].tolist() == [3, 0, 4, 1, 2]
    assert r["tier"].tolist() == [0, 2, 3, 0, 1]          # GPU: p3 p0 (5); next: p4 (4); next: p1 (1); p2 waits
    assert r["bounds"].tolist() == [2, 3, 4] and r["used"].tolist() == [5, 4, 1]


@pytest.mark.parametrize("n", [0, 1, 9, 200, 3000])
def test_two_tiers_is_rank_partition_and_restatement_agrees(n):
    rng = np.random.default_rng(n + 5)
    for _ in range(10):
        iota, s, prev, cg, cc = _rand_case(rng, n)
        two = oracle.rank_partition_tiers(iota, s, [cg, cc])
        ref = oracle.rank_partition(iota, s, None, cg, cc)
        assert np.array_equal(two["order"], ref["order"]) and np.array_equal(two["tier"], ref["tier"])
        assert np.array_equal(two["bounds"], ref["bounds"]) and np.array_equal(two["used"], ref["used"])
        caps = rng.integers(0, max(2, int(np.sum(s)) // 2 + 2), int(rng.integers(1, 9)))
        a, b = oracle.rank_partition_tiers(iota, s, caps), oracle_np.rank_partition_tiers(iota, s, caps)
        for k in ("order", "tier", "bounds", "used"):
            assert np.array_equal(a[k], b[k]), k


def test_three_tiers_brute_force():
    """All 4^n maps programs -> {0, 1, 2, waiting}: capacities respected, order-consistent (a
    program in an earlier tier is busier than every program in a later one); the lexicographic
    maximum of the tier sizes is unique and is the oracle's answer."""
    rng = np.random.default_rng(2)
    for _ in range(40):
        n = int(rng.integers(1, 7))
        iota = (np.round(rng.random(n) * 4) / 4).astype(np.float32)
        s = rng.integers(1, 6, n).astype(np.int32)
        caps = rng.integers(0, 9, 3)
        pos = np.empty(n, np.int64); pos[oracle_np.rank(iota)] = np.arange(n)
        best, best_maps = None, []
        for t in itertools.product(range(4), repeat=n):
            t = np.array(t)
            if any(s[t == k].sum() > caps[k] for k in range(3)):
                continue
            if any(t[a] < t[b] and pos[a] > pos[b] for a in range(n) for b in range(n)):
                continue
            key = tuple(int((t == k).sum()) for k in range(3))
            if best is None or key > best:
                best, best_maps = key, [t]
            elif key == best:
                best_maps.append(t)
        assert len(best_maps) == 1
        assert oracle.rank_partition_tiers(iota, s, caps)["tier"].tolist() == best_maps[0].tolist()


def test_bad_arguments():
    with pytest.raises(ValueError):
        oracle.rank_partition_tiers([0.1], [1], [])
    with pytest.raises(ValueError):
        oracle.rank_partition_tiers([0.1], [1], [1] * 9)
    with pytest.raises(ValueError):
        oracle.rank_partition_tiers([0.1], [1], [-1])


def test_move_lists_generalise_the_two_tier_lists():
    """With T = 2 the down list is demote + drop merged in rank order (most idle first) and the up
    list is promote + admit + reserve (least idle first) of the pinned two-tier oracle; for any T
    the C loops and the numpy masks agree, and the lists are exactly the programs whose tier
    changed."""
    rng = np.random.default_rng(12)
    for n in (0, 1, 8, 100, 2000):
        for _ in range(8):
            iota, s, prev, cg, cc = _rand_case(rng, n)
            prev = rng.integers(0, 4, n).astype(np.uint8) if prev is None else prev
            two = oracle.rank_partition_tiers(iota, s, [cg, cc], prev)
            ref = oracle.rank_partition(iota, s, prev, cg, cc)
            pos = np.empty(n, np.int64); pos[ref["order"]] = np.arange(n)
            down = np.concatenate([ref["lists"][0], ref["lists"][2]]); down = down[np.argsort(-pos[down], kind="stable")]
            up = np.concatenate([ref["lists"][1], ref["lists"][3], ref["lists"][4]]); up = up[np.argsort(pos[up], kind="stable")]
            assert np.array_equal(two["moves"][0], down) and np.array_equal(two["moves"][1], up)
            T = int(rng.integers(1, 9))
            caps = rng.integers(0, max(2, int(np.sum(s)) // T + 2), T)
            pv = rng.integers(0, T + 2, n).astype(np.uint8)
            a, b = oracle.rank_partition_tiers(iota, s, caps, pv), oracle_np.rank_partition_tiers(iota, s, caps, pv)
            for k in range(2):
                assert np.array_equal(a["moves"][k], b["moves"][k])
            changed = set(np.flatnonzero(a["tier"] != np.minimum(pv, T)).tolist())
            assert changed == set(a["moves"][0].tolist()) | set(a["moves"][1].tolist())
            assert len(changed) == a["moves"][0].size + a["moves"][1].size


# ------------------------------------------------------------------------------------------------
# the arena <-> arena mover and whole three-pool epochs (an intermediate tier)
# ------------------------------------------------------------------------------------------------
def test_move_slots_is_a_per_page_copy():
    rng = np.random.default_rng(3)
    page = 48
    src = rng.integers(0, 256, 9 * page, dtype=np.uint8)
    dst0 = rng.integers(0, 256, 7 * page, dtype=np.uint8)
    a, b = np.array([8, 0, 3, 3], np.int32), np.array([1, 6, 0, 4], np.int32)
    dst = dst0.copy()
    oracle.move_slots(page, src, dst, a, b)
    want = dst0.copy()
    for j in range(len(a)):                                  # byte by byte
        for x in range(page):
            want[b[j] * page + x] = src[a[j] * page + x]
    assert np.array_equal(dst, want)
    dst2 = dst0.copy()
    oracle_np.move_slots(page, src, dst2, a, b)              # fancy-index restatement
    assert np.array_equal(dst2, want)
    untouched = np.setdiff1d(np.arange(7), b)
    assert np.array_equal(dst.reshape(7, page)[untouched], dst0.reshape(7, page)[untouched])
    back = np.zeros_like(src)                                # round trip into other slots
    oracle.move_slots(page, dst, back, b[:3], np.array([2, 5, 7], np.int32))
    assert np.array_equal(back.reshape(9, page)[[2, 5, 7]], src.reshape(9, page)[a[:3]])
    with pytest.raises(ValueError):
        oracle.move_slots(page, src, dst, np.array([9], np.int32), np.array([0], np.int32))
    with pytest.raises(ValueError):
        oracle.move_slots(page, src, dst, np.array([0], np.int32), np.array([7], np.int32))
    oracle.move_slots(page, src, dst, np.zeros(0, np.int32), np.zeros(0, np.int32))


def test_move_slots_equals_demote_of_a_one_layer_pool():
    """An arena described as a pool of ONE layer whose chunk is a whole page is the same bytes, so
    the arena <-> arena move must equal the (already pinned) pool -> arena mover on that view."""
    rng = np.random.default_rng(4)
    page, S1, S2 = 96, 20, 30
    src = rng.integers(0, 256, S1 * page, dtype=np.uint8)
    d1 = rng.integers(0, 256, S2 * page, dtype=np.uint8)
    d2 = d1.copy()
    a = rng.permutation(S1)[:12].astype(np.int32)
    b = rng.permutation(S2)[:12].astype(np.int32)
    oracle.move_slots(page, src, d1, a, b)
    oracle.demote(1, page, src, d2, a, b)
    assert np.array_equal(d1, d2)


def three_pool_epochs(cfg, seed, pool_ids, caps, epochs, on_epoch=None):
    """Whole epochs of a three-tier hierarchy on the ORACLE side: oracle_rank_partition_tiers decides,
    workload.SimTiers turns the move lists into tables, the oracle's memcpy movers carry them out on
    byte mirrors of the three pools.  Yields nothing; calls on_epoch(e, sim, plan, res, mirrors)."""
    from paper_2606_00866_b200 import workload as W
    sh = cfg.shape
    sim = W.SimTiers(cfg, seed, pool_ids, caps)
    pool = np.zeros(sh.n_layers * pool_ids[0] * sh.chunk_bytes, np.uint8)
    mid = np.zeros(pool_ids[1] * sh.page_bytes, np.uint8)
    host = np.zeros(pool_ids[2] * sh.page_bytes, np.uint8)
    for e in range(epochs):
        plan = sim.begin_epoch()
        res = oracle.rank_partition_tiers(plan.iota, plan.kv_pages, caps, plan.prev_tier)
        sim.apply_placement(res["tier"], res["moves"])
        oracle_apply_moves(plan.ops, sh, pool, mid, host)
        sim.end_epoch()
        pv = pool.reshape(sh.n_layers, pool_ids[0], sh.chunk_bytes)
        for uid, first, pages in plan.fills:
            for j, g in enumerate(pages):
                pv[:, g] = W.page_content(seed, uid, first + j, sh)
        if on_epoch:
            on_epoch(e, sim, plan, res, (pool, mid, host))
    return sim, (pool, mid, host)


def oracle_apply_moves(ops, sh, pool, mid, host):
    arenas = {1: mid, 2: host}
    for op in ops:
        if op[0] != "move":
            continue
        _, p, frm, to, src, dst = op
        if frm == 0:
            oracle.demote(sh.n_layers, sh.chunk_bytes, pool, arenas[to], src, dst)
        elif to == 0:
            oracle.promote(sh.n_layers, sh.chunk_bytes, pool, arenas[frm], src, dst)
        else:
            oracle.move_slots(sh.page_bytes, arenas[frm], arenas[to], src, dst)


def _check_resident_against_generator(sim, mirrors, seed):
    """Every byte of every resident page, in whichever pool it lives, equals the counter-based
    generator G(seed, uid, logical page): a check that needs no second mover."""
    from paper_2606_00866_b200 import workload as W
    sh = sim.cfg.shape
    pool, mid, host = mirrors
    views = [pool.reshape(sh.n_layers, -1, sh.chunk_bytes), mid.reshape(-1, sh.n_layers, sh.chunk_bytes),
             host.reshape(-1, sh.n_layers, sh.chunk_bytes)]
    n = 0
    for t, tri in enumerate(sim.resident()):
        for uid, first, ids in tri:
            for j, i in enumerate(ids):
                want = W.page_content(seed, uid, first + j, sh)
                have = views[0][:, i] if t == 0 else views[t][i]
                assert np.array_equal(have, want), (t, uid, j)
                n += 1
    return n


def _small_cfg2():
    """cfg 2's scaled twin (same programs, page counts and trace) with a small KV shape, so that the
    byte-level checks of these CPU pins stay fast: 16 KiB pages instead of 2 MiB."""
    from dataclasses import replace
    from paper_2606_00866_b200 import workload as W
    return replace(W.get_config(2, 128), shape=W.KVShape(4, 2, 32, 16))


@pytest.mark.parametrize("mid_ids,mid_slack", [(160, None), (120, 0)])
def test_three_pool_epochs_keep_every_resident_page_intact(mid_ids, mid_slack):
    """mid_slack = physical middle slots the ranker is NOT given (None: one largest program).  With no
    slack at all the planner must split epochs into phases separated by joins (ids freed in a phase
    are not reused before the next join); the bytes must come out right either way."""
    cfg = _small_cfg2()
    mid_cap = mid_ids - (cfg.max_program_pages if mid_slack is None else mid_slack)
    pool_ids = [cfg.gpu_pool_pages, mid_ids, cfg.cpu_pool_pages]
    caps = [cfg.cap_gpu_pages, mid_cap, cfg.cap_cpu_pages]
    seen = {"pairs": set(), "pages": 0, "joins": 0}

    def on_epoch(e, sim, plan, res, mirrors):
        seen["joins"] += sum(1 for op in plan.ops if op[0] == "sync_all")
        for op in plan.ops:
            if op[0] == "move":
                seen["pairs"].add((op[2], op[3]))
        # capacities of the partition hold for what is physically resident too
        for t in range(3):
            assert sum(int(x[2].size) for x in sim.resident()[t]) <= pool_ids[t]
        if e % 5 == 4:
            seen["pages"] += _check_resident_against_generator(sim, mirrors, 866)

    three_pool_epochs(cfg, 866, pool_ids, caps, 40, on_epoch)
    assert seen["pages"] > 500
    # the hierarchy was really exercised: bytes went down and up between all neighbouring pairs
    assert {(0, 1), (1, 0), (1, 2)} <= seen["pairs"], seen["pairs"]
    if mid_slack == 0:
        assert seen["joins"] >= 5, "a middle pool with no slack must force mid-epoch joins"


def test_three_pool_epochs_with_an_empty_middle_tier_are_the_two_pool_epochs():
    """T = 3 with capacity 0 in the middle reduces to the pinned two-tier path: the same tiers and
    the same programs moving the same way every epoch (down = demote + drop, up = promote + admit +
    reserve), and the same logical bytes for every program afterwards."""
    from paper_2606_00866_b200 import workload as W
    cfg = _small_cfg2()
    seed = 867
    sim2 = W.Sim(cfg, seed)
    two = []

    for e in range(25):
        plan = sim2.begin_epoch()
        r2 = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        sim2.apply_placement(r2["tier"], r2["lists"])
        sim2.end_epoch()
        two.append((r2, plan))

    def on_epoch(e, sim, plan, res, mirrors):
        r2, plan2 = two[e]
        assert np.array_equal(plan.iota, plan2.iota) and np.array_equal(plan.kv_pages, plan2.kv_pages)
        t3 = res["tier"].copy()
        assert not np.any(t3 == 1)                           # nobody fits a tier of capacity 0 (sizes > 0)
        assert np.array_equal(np.where(t3 == 2, 1, np.where(t3 == 3, 2, t3)), r2["tier"])
        moved3 = {(op[1], op[2], op[3]) for op in plan.ops if op[0] == "move"}
        moved2 = {(op[2], 0, 2) for op in plan2.ops if op[0] == "demote"} | \
                 {(op[2], 2, 0) for op in plan2.ops if op[0] == "promote"}
        assert moved3 == moved2, e
        assert plan.demote_pages == plan2.demote_pages and plan.promote_pages == plan2.promote_pages

    sim3, mirrors = three_pool_epochs(cfg, seed, [cfg.gpu_pool_pages, 8, cfg.cpu_pool_pages],
                                      [cfg.cap_gpu_pages, 0, cfg.cap_cpu_pages], 25, on_epoch)
    assert _check_resident_against_generator(sim3, mirrors, seed) > 100
    assert not mirrors[1].any()                              # nothing ever touched the middle pool
