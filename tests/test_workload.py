"""Host logic: the seeded input generators and the epoch planner (no method arithmetic there),
and the oracle driven over whole synthetic runs (brute force on every cfg-1 epoch)."""
import os

import numpy as np
import pytest

import oracle
from paper_2606_00866_b200 import workload as W
from test_oracle_pins import check_invariants, check_lists

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_eq1_closed_forms():
    for line in open(os.path.join(GOLD, "eq1_examples.txt")):
        if line.startswith("#") or not line.strip():
            continue
        r, a, want = [x.split() for x in line.split("|")]
        got = W.windowed_idleness(np.array(r, float), np.array(a, float))
        assert got == np.float32(float(want[0]))
    assert np.isnan(W.windowed_idleness(np.zeros(5), np.zeros(5)))


def test_eq1_responsive_and_outlier_robust():
    # an ongoing long tool call soon dominates; one outlier among k=5 is diluted
    base_r, base_a = [4.0] * 4, [1.0] * 4
    prev = 0.0
    for elapsed in (1, 10, 60, 600):
        i = W.windowed_idleness(np.array(base_r + [4.0]), np.array(base_a + [elapsed]))
        assert i > prev
        prev = i
    assert prev > 0.95
    assert W.windowed_idleness(np.array([4.0] * 5), np.array([1, 1, 1, 1, 8.0])) < 0.4


def test_config_shapes_match_baseline_json():
    want = {1: (8 << 10, 16 << 10, 64, 256), 2: (64 << 10, 2 << 20, 30720, 65536),
            3: (64 << 10, 4 << 20, 20480, 40960), 4: (128 << 10, 10 << 20, 10240, 20480),
            5: (64 << 10, 2 << 20, 30720, 65536)}
    for i, (chunk, page, gp, cp) in want.items():
        c = W.get_config(i)
        assert (c.shape.chunk_bytes, c.shape.page_bytes, c.gpu_pool_pages, c.cpu_pool_pages) == (chunk, page, gp, cp)
    c = W.get_config(3, scale=16)
    assert c.gpu_pool_pages == 1280 and c.shape == W.get_config(3).shape and c.n_programs == 128


def test_trace_is_seed_deterministic_and_in_range():
    cfg = W.get_config(2, scale=16)
    a, b = W.Trace(cfg, 866), W.Trace(cfg, 866)
    tier = np.zeros(cfg.n_programs, np.uint8)
    for _ in range(30):
        ia, ta, ra = a.advance(tier)
        ib, tb, rb = b.advance(tier)
        assert np.array_equal(ia, ib) and np.array_equal(ta, tb) and np.array_equal(ra, rb)
        assert ia.dtype == np.float32 and ((ia >= 0) & (ia <= 1)).all()
        assert (ta >= cfg.ctx_lo).all() and (ta <= cfg.ctx_hi).all()
    c = W.Trace(cfg, 867)
    assert not np.array_equal(c.advance(tier)[0], ia)


def test_gated_time_is_excluded():
    # a program that is never on the GPU never accrues reasoning time
    cfg = W.get_config(1)
    t = W.Trace(cfg, 1)
    tier = np.full(cfg.n_programs, W.TIER_WAIT, np.uint8)
    first, _, _ = t.advance(tier)
    for _ in range(50):
        iota, _, rep = t.advance(tier)
    assert not rep.any() and np.array_equal(iota, first)


def test_page_content_generator():
    sh = W.KVShape(2, 2, 64, 16)
    a = W.page_content(866, 3, 5, sh)
    assert a.shape == (2, sh.chunk_bytes) and a.dtype == np.uint8
    assert np.array_equal(a, W.page_content(866, 3, 5, sh))
    assert not np.array_equal(a, W.page_content(866, 3, 6, sh))
    assert not np.array_equal(a, W.page_content(866, 4, 5, sh))
    assert not np.array_equal(a[0], a[1])
    # bf16 values ~ N(0,1)
    v = (a.reshape(-1).view(np.uint16).astype(np.uint32) << 16).view(np.float32)
    assert abs(v.mean()) < 0.05 and 0.9 < v.std() < 1.1


def _run(cfg, seed, epochs, brute=False, mirror=False):
    sim = W.Sim(cfg, seed)
    sh = cfg.shape
    if mirror:
        pool = np.zeros(sh.n_layers * cfg.gpu_pool_pages * sh.chunk_bytes, np.uint8)
        arena = np.zeros(cfg.cpu_pool_pages * sh.page_bytes, np.uint8)
    seen = np.zeros(3, int)
    moved = 0
    for _ in range(epochs):
        plan = sim.begin_epoch()
        r = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier,
                                  cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        check_invariants(plan.iota, plan.kv_pages, cfg.cap_gpu_pages, cfg.cap_cpu_pages, r)
        check_lists(plan.prev_tier, r)
        if brute:
            b = oracle.bruteforce_partition(plan.iota, plan.kv_pages, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
            assert b["n_best"] == 1 and np.array_equal(b["tier"], r["tier"])
        sim.apply_placement(r["tier"], r["lists"])
        if mirror:
            for op in plan.ops:
                if op[0] == "demote":
                    oracle.demote(sh.n_layers, sh.chunk_bytes, pool, arena, op[3], op[4])
                elif op[0] == "promote":
                    oracle.promote(sh.n_layers, sh.chunk_bytes, pool, arena, op[3], op[4])
        sim.end_epoch()
        if mirror:
            pv = pool.reshape(sh.n_layers, cfg.gpu_pool_pages, sh.chunk_bytes)
            for uid, first, pages in plan.fills:
                for j, g in enumerate(pages):
                    pv[:, g] = W.page_content(seed, uid, first + j, sh)
            # every resident logical page holds exactly its generated content
            av = arena.reshape(cfg.cpu_pool_pages, sh.n_layers, sh.chunk_bytes)
            for p in range(cfg.n_programs):
                uid = int(sim.trace.uid[p])
                for j, g in enumerate(sim.gpu_pages[p]):
                    assert np.array_equal(pv[:, g], W.page_content(seed, uid, j, sh))
                for j, h in enumerate(sim.host_slots[p]):
                    assert np.array_equal(av[h], W.page_content(seed, uid, j, sh))
        # no page / slot owned twice; tiers own what they should
        gp = np.concatenate(sim.gpu_pages)
        hs = np.concatenate(sim.host_slots)
        assert len(set(gp.tolist())) == gp.size and len(set(hs.tolist())) == hs.size
        assert not sim.gpu_alloc.free[gp].any() and not sim.cpu_alloc.free[hs].any()
        assert sim.gpu_alloc.free.sum() + gp.size == cfg.gpu_pool_pages
        assert sim.cpu_alloc.free.sum() + hs.size == cfg.cpu_pool_pages
        for p in range(cfg.n_programs):
            if sim.tier[p] == W.TIER_GPU:
                assert sim.gpu_pages[p].size == plan.kv_pages[p] and sim.host_slots[p].size == 0
            elif sim.tier[p] == W.TIER_CPU:
                assert sim.gpu_pages[p].size == 0 and sim.host_slots[p].size <= plan.kv_pages[p]
            else:
                assert sim.gpu_pages[p].size == 0 and sim.host_slots[p].size == 0
        seen += np.bincount(sim.tier, minlength=3)
        moved += plan.demote_pages + plan.promote_pages
    return seen, moved


@pytest.mark.parametrize("seed", [866, 867, 868])
def test_cfg1_oracle_run_bruteforce_every_epoch_with_byte_mirror(seed):
    cfg = W.get_config(1)
    seen, moved = _run(cfg, seed, cfg.epochs, brute=True, mirror=True)
    assert seen[0] > 0


@pytest.mark.parametrize("idx,scale,epochs", [(2, 32, 60), (3, 32, 40), (4, 32, 30), (5, 32, 20)])
def test_scaled_twins_oracle_run(idx, scale, epochs):
    cfg = W.get_config(idx, scale=scale)
    seen, moved = _run(cfg, 866, epochs)
    assert seen.min() > 0 and moved > 0          # all three tiers occur and pages move


def test_cfg3_busy_fraction_moves_the_boundary():
    frac = []
    for f in (0.25, 0.5, 0.75):
        cfg = W.get_config(3, scale=32, f_busy=f)
        t = W.Trace(cfg, 866)
        tier = np.zeros(cfg.n_programs, np.uint8)
        for _ in range(40):
            iota, _, _ = t.advance(tier)
        frac.append(float((iota < 0.5).mean()))
    assert frac[0] < frac[1] < frac[2]


def test_alloc_run_gives_one_contiguous_clean_run_or_falls_back():
    a = W.IdAllocator(32, None)
    x, _ = a.alloc(10)                       # ids 0..9
    a.release(x[2:5])                        # hole of 3 at 2..4
    a.release(x[7:9], tag=3)                 # dirty hole at 7..8 (not yet reusable)
    r, dep = a.alloc_run(3)
    assert r.tolist() == [2, 3, 4] and dep == 0
    r, _ = a.alloc_run(5)                    # first clean run of >= 5 starts at 10
    assert r.tolist() == [10, 11, 12, 13, 14]
    r, _ = a.alloc_run(17)                   # exactly the rest
    assert r.tolist() == list(range(15, 32))
    a.release(np.array([0, 1, 20, 21, 30]))
    r, _ = a.alloc_run(4)                    # no run of 4: fragments, lowest clean ids
    assert sorted(r.tolist()) == [0, 1, 20, 21]
    with pytest.raises(MemoryError):
        a.alloc_run(5)
    assert a.alloc_run(0)[0].size == 0


def test_plan_calls_keeps_order_bytes_and_dependencies():
    """The merged call lists carry exactly the plan's pages, each direction in plan order, and a
    promotion that lands in pages a demotion vacates is issued after the call that carries it."""
    import oracle
    cfg = W.get_config(3, 32, 0.5)          # the config whose promotions do depend on demotions
    sim = W.Sim(cfg, 866)
    seen_dep = seen_split = 0
    for e in range(120):
        plan = sim.begin_epoch()
        res = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        sim.apply_placement(res["tier"], res["lists"])
        for merge in (True, False):
            steps, need = W.plan_calls(plan, merge=merge)
            dem_ops = [op for op in plan.ops if op[0] == "demote"]
            pro_ops = [op for op in plan.ops if op[0] == "promote"]
            d_steps = [st for st in steps if st[0] == "d"]
            p_steps = [st for st in steps if st[0] == "p"]
            cat = lambda xs: np.concatenate(xs) if xs else np.zeros(0, np.int32)
            assert np.array_equal(cat([st[1] for st in d_steps]), cat([op[3] for op in dem_ops]))
            assert np.array_equal(cat([st[2] for st in d_steps]), cat([op[4] for op in dem_ops]))
            # promotions: same multiset of (slot, page) pairs, and plan order inside every dependency class
            got = np.stack([cat([st[1] for st in p_steps]), cat([st[2] for st in p_steps])]) if p_steps else np.zeros((2, 0))
            want = np.stack([cat([op[3] for op in pro_ops]), cat([op[4] for op in pro_ops])]) if pro_ops else np.zeros((2, 0))
            assert sorted(map(tuple, got.T.tolist())) == sorted(map(tuple, want.T.tolist()))
            carried = set()
            for st in steps:
                if st[0] == "d":
                    carried.update(st[4])
                elif st[0] == "p" and st[4] > 0:
                    assert st[4] in carried, "a dependent promotion was issued before its demotion"
                elif st[0] == "sync":
                    carried.clear()
            assert need == any(op[5] > 0 for op in pro_ops)
            if not merge:
                assert len(d_steps) == len(dem_ops) and len(p_steps) == len(pro_ops)
        seen_dep += any(op[0] == "promote" and op[5] > 0 for op in plan.ops)
        per_prog = {}
        for op in plan.ops:
            if op[0] == "promote":
                per_prog.setdefault(op[2], []).append(op)
        for ops in per_prog.values():          # a split promotion covers its program's pages once, in order
            if len(ops) > 1:
                seen_split += 1
                firsts = [op[6] for op in ops]
                assert firsts == sorted(firsts) and firsts[0] == 0
                assert all(firsts[i] + len(ops[i][3]) == firsts[i + 1] for i in range(len(ops) - 1))
        sim.end_epoch()
    assert seen_dep > 0 and seen_split > 0, "the trace never produced a dependent promotion"


def test_two_tier_planner_never_aliases_pages_without_a_ticket():
    """What the movers rely on: within an epoch, a promotion lands either in pages nothing is
    reading (free before the epoch's moves began, or freed before the last join) or in pages freed
    by exactly the demotion it names as its dependency; a demotion writes slots nothing reads."""
    import oracle
    for idx, scale, fb in ((3, 32, 0.5), (2, 64, None), (5, 64, None)):
        cfg = W.get_config(idx, scale, fb)
        sim = W.Sim(cfg, 867)
        for e in range(60):
            plan = sim.begin_epoch()
            res = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
            sim.apply_placement(res["tier"], res["lists"])
            freed_by = {}                       # gpu page -> demote number that vacates it (since the last join)
            slots_read = set()                  # host slots a promotion of this phase reads
            slots_written = set()
            for op in plan.ops:
                if op[0] == "sync_all":
                    freed_by.clear(); slots_read.clear(); slots_written.clear()
                elif op[0] == "demote":
                    for g in op[3]:
                        assert int(g) not in freed_by
                        freed_by[int(g)] = op[1]
                    assert not (set(map(int, op[4])) & (slots_read | slots_written)), "a demotion writes a slot in use"
                    slots_written.update(map(int, op[4]))
                else:
                    deps = {freed_by[int(g)] for g in op[4] if int(g) in freed_by}
                    assert deps <= ({op[5]} if op[5] > 0 else set()), (e, deps, op[5])
                    assert not (set(map(int, op[3])) & slots_written), "a promotion reads a slot written this phase"
                    slots_read.update(map(int, op[3]))
            sim.end_epoch()
            # every program's pages / slots are its own
            allg = np.concatenate([p for p in sim.gpu_pages if p.size] or [np.zeros(0, np.int32)])
            allh = np.concatenate([p for p in sim.host_slots if p.size] or [np.zeros(0, np.int32)])
            assert np.unique(allg).size == allg.size and np.unique(allh).size == allh.size
            assert allg.size <= cfg.gpu_pool_pages and allh.size <= cfg.cpu_pool_pages


def test_tier_planner_never_reuses_an_id_freed_in_the_same_phase():
    """SimTiers promises the three pair-movers that no id freed by a move is handed out again before
    the next join, and that every program's ids stay disjoint in every pool."""
    import oracle
    cfg = W.get_config(2, 64)
    for mid_ids, slack in ((cfg.gpu_pool_pages // 2, cfg.max_program_pages // 2), (cfg.gpu_pool_pages // 3, 0)):
        pool_ids = [cfg.gpu_pool_pages, mid_ids, cfg.cpu_pool_pages]
        caps = [cfg.cap_gpu_pages, mid_ids - slack, cfg.cap_cpu_pages]
        sim = W.SimTiers(cfg, 868, pool_ids, caps)
        for e in range(50):
            plan = sim.begin_epoch()
            res = oracle.rank_partition_tiers(plan.iota, plan.kv_pages, caps, plan.prev_tier)
            sim.apply_placement(res["tier"], res["moves"])
            freed = [set(), set(), set()]
            for op in plan.ops:
                if op[0] == "sync_all":
                    freed = [set(), set(), set()]
                else:
                    _, p, frm, to, src, dst = op
                    assert frm != to and len(src) == len(dst)
                    assert not (set(map(int, dst)) & freed[to]), (e, "id reused before a join")
                    freed[frm].update(map(int, src))
            sim.end_epoch()
            for t, tri in enumerate(sim.resident()):
                ids = np.concatenate([x[2] for x in tri]) if tri else np.zeros(0, np.int32)
                assert np.unique(ids).size == ids.size and ids.size <= pool_ids[t]
                assert ids.size == 0 or (ids.min() >= 0 and ids.max() < pool_ids[t])
            # the label and the location agree for every program that holds bytes
            for p in range(cfg.n_programs):
                if sim.where[p] >= 0:
                    assert sim.where[p] == sim.tier[p], (e, p)
