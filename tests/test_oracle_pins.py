"""Pins for the CPU oracle: it is checked against things that are not itself -- brute-force
enumeration, numpy library routines, closed forms, a hand-worked example and the paper's
invariants -- so that a dropped term, a wrong sign or index, or a
transposed operand fails at least one of them."""
import os

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import oracle
from oracle import oracle_np

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    d = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        d[k] = v
    return d


def check_invariants(iota, s, cap_g, cap_c, r):
    """Ordering, capacity and maximality -- stated without the oracle's own loop."""
    n = len(s)
    order, tier, (bg, bc) = r["order"], r["tier"], r["bounds"]
    assert sorted(order.tolist()) == list(range(n))
    # ranking is the total order
    f = np.asarray(iota, np.float32)
    for a, b in zip(order[:-1], order[1:]):
        fa, fb = f[a], f[b]
        if np.isnan(fa):
            assert np.isnan(fb) and a < b
        elif not np.isnan(fb):
            assert fa < fb or (fa == fb and a < b)
    # tiers are contiguous rank ranges: every GPU program is busier than every CPU program
    t_by_rank = tier[order]
    assert (np.diff(t_by_rank.astype(int)) >= 0).all()
    assert (t_by_rank == 0).sum() == bg and (t_by_rank <= 1).sum() == bc
    # capacity
    ug, uc = int(s[tier == 0].sum()), int(s[tier == 1].sum())
    assert ug <= cap_g and uc <= cap_c
    assert (ug, uc) == tuple(int(x) for x in r["used"])
    # maximality ("filling each tier to capacity")
    if bg < n:
        assert ug + s[order[bg]] > cap_g
    if bc < n:
        assert uc + s[order[bc]] > cap_c


def check_lists(prev, r):
    n = len(prev)
    tier, order, lists = r["tier"], r["order"], r["lists"]
    prev = np.where(np.asarray(prev) > 2, 2, prev)
    rank_of = np.empty(n, int)
    rank_of[order] = np.arange(n)
    want = [(0, 1), (1, 0), None, (2, 0), (2, 1)]
    seen = set()
    for k, lst in enumerate(lists):
        for p in lst:
            assert p not in seen
            seen.add(int(p))
            if want[k] is None:
                assert prev[p] != 2 and tier[p] == 2
            else:
                assert (prev[p], tier[p]) == want[k]
        ranks = rank_of[lst]
        if k in (0, 2):
            assert (np.diff(ranks) < 0).all()      # most idle first
        else:
            assert (np.diff(ranks) > 0).all()      # least idle first
    moved = {p for p in range(n) if prev[p] != tier[p]}
    assert moved == seen


# ---------------------------------------------------------------- hand-worked golden example
def test_handworked_example():
    g = _gold("placement_handworked.txt")
    iota = np.array(g["iota"], np.float32)
    s = np.array(g["pages"], np.int32)
    prev = np.array(g["prev_tier"], np.uint8)
    cg, cc = map(int, g["cap"])
    for impl in (oracle.rank_partition, oracle_np.rank_partition):
        r = impl(iota, s, prev, cg, cc)
        assert r["order"].tolist() == list(map(int, g["order"]))
        assert r["tier"].tolist() == list(map(int, g["tier"]))
        assert r["bounds"].tolist() == list(map(int, g["bounds"]))
        assert r["used"].tolist() == list(map(int, g["used"]))
        for k, name in enumerate(["demote", "promote", "drop", "admit", "reserve"]):
            assert r["lists"][k].tolist() == list(map(int, g[name])), name
    b = oracle.bruteforce_partition(iota, s, cg, cc)
    assert b["tier"].tolist() == list(map(int, g["tier"])) and b["n_best"] == 1


# ---------------------------------------------------------------- brute force
small_case = st.integers(0, 9).flatmap(lambda n: st.tuples(
    st.lists(st.sampled_from([0.0, -0.0, 0.1, 0.25, 0.5, 0.5, 0.9, 1.0, 7.0, float("inf"),
                              float("-inf"), float("nan")]), min_size=n, max_size=n),
    st.lists(st.integers(0, 6), min_size=n, max_size=n),
    st.integers(0, 20), st.integers(0, 20)))


@settings(max_examples=300, deadline=None)
@given(small_case)
def test_bruteforce_equals_scan(case):
    iota, s, cg, cc = case
    iota, s = np.array(iota, np.float32), np.array(s, np.int32)
    r = oracle.rank_partition(iota, s, None, cg, cc)
    b = oracle.bruteforce_partition(iota, s, cg, cc)
    assert b["n_best"] == 1                       # the maximiser is unique
    assert b["tier"].tolist() == r["tier"].tolist()
    assert b["bounds"].tolist() == r["bounds"].tolist()
    check_invariants(iota, s, cg, cc, r)


def test_bruteforce_random_floats():
    rng = np.random.default_rng(1)
    for _ in range(200):
        n = int(rng.integers(1, 9))
        iota = rng.random(n).astype(np.float32)
        iota[rng.random(n) < 0.3] = iota[0]       # ties
        s = rng.integers(0, 30, n).astype(np.int32)
        cg, cc = int(rng.integers(0, 60)), int(rng.integers(0, 60))
        r = oracle.rank_partition(iota, s, None, cg, cc)
        b = oracle.bruteforce_partition(iota, s, cg, cc)
        assert b["n_best"] == 1 and b["tier"].tolist() == r["tier"].tolist()


# ---------------------------------------------------------------- numpy restatement
def _rand_case(rng, n):
    kind = rng.integers(0, 4)
    if kind == 0:
        iota = rng.random(n)
    elif kind == 1:
        iota = rng.lognormal(0, 1, n)
    elif kind == 2:
        iota = rng.integers(0, 4, n) / 4.0                   # heavy ties
    else:
        iota = rng.standard_normal(n)
    iota = iota.astype(np.float32)
    special = np.array([0.0, -0.0, np.inf, -np.inf, np.nan], np.float32)
    m = rng.random(n) < 0.05
    iota[m] = special[rng.integers(0, 5, m.sum())]
    s = rng.integers(0, 5000, n).astype(np.int32)
    s[rng.random(n) < 0.05] = 0
    tot = int(s.sum())
    cg = int(rng.integers(0, tot + 2)) if rng.random() < 0.9 else tot * 2
    cc = int(rng.integers(0, tot + 2))
    prev = rng.integers(0, 3, n).astype(np.uint8)
    return iota, s, prev, cg, cc


def test_c_equals_numpy_restatement():
    rng = np.random.default_rng(2)
    for n in [0, 1, 2, 3, 8, 64, 128, 256, 1000, 4096, 5000] * 3:
        iota, s, prev, cg, cc = _rand_case(rng, n)
        a = oracle.rank_partition(iota, s, prev, cg, cc)
        b = oracle_np.rank_partition(iota, s, prev, cg, cc)
        for k in ("order", "tier", "bounds", "used"):
            assert np.array_equal(a[k], b[k]), (n, k)
        for la, lb in zip(a["lists"], b["lists"]):
            assert np.array_equal(la, lb)
        check_invariants(iota, s, cg, cc, a)
        check_lists(prev, a)


def test_sort_reduces_to_library_argsort():
    rng = np.random.default_rng(3)
    iota = rng.random(1000).astype(np.float32)
    s = np.ones(1000, np.int32)
    r = oracle.rank_partition(iota, s, None, 10, 10)
    assert np.array_equal(r["order"], np.argsort(iota, kind="stable"))


# ---------------------------------------------------------------- closed forms
def test_all_equal_idleness_is_identity_and_decreasing_is_reversal():
    n = 100
    s = np.ones(n, np.int32)
    r = oracle.rank_partition(np.full(n, 0.5, np.float32), s, None, 10, 10)
    assert r["order"].tolist() == list(range(n))
    r = oracle.rank_partition(np.linspace(1, 0, n).astype(np.float32), s, None, 10, 10)
    assert r["order"].tolist() == list(range(n))[::-1]


def test_signed_zero_ties_and_nan_last():
    iota = np.array([np.nan, 0.0, -0.0, np.inf, -np.inf, np.nan, 0.0], np.float32)
    r = oracle.rank_partition(iota, np.ones(7, np.int32), None, 7, 0)
    assert r["order"].tolist() == [4, 1, 2, 6, 3, 0, 5]


@pytest.mark.parametrize("n,size,cg,cc", [(10, 3, 10, 7), (10, 3, 9, 9), (5, 4, 100, 100),
                                          (7, 2, 0, 5), (7, 2, 5, 0), (6, 1, 3, 3)])
def test_equal_sizes_closed_form(n, size, cg, cc):
    rng = np.random.default_rng(n)
    r = oracle.rank_partition(rng.random(n).astype(np.float32), np.full(n, size, np.int32), None, cg, cc)
    bg = min(n, cg // size)
    bc = bg + min(n - bg, cc // size)
    assert r["bounds"].tolist() == [bg, bc]
    assert r["used"].tolist() == [bg * size, (bc - bg) * size]


def test_capacity_extremes():
    rng = np.random.default_rng(5)
    iota, s = rng.random(50).astype(np.float32), rng.integers(1, 9, 50).astype(np.int32)
    r = oracle.rank_partition(iota, s, None, 0, 0)
    assert (r["tier"] == 2).all() and r["bounds"].tolist() == [0, 0]
    r = oracle.rank_partition(iota, s, None, int(s.sum()), 0)
    assert (r["tier"] == 0).all()
    r = oracle.rank_partition(iota, s, None, 0, int(s.sum()))
    assert (r["tier"] == 1).all()
    r = oracle.rank_partition(iota, s, None, int(s.sum()) - 1, 1 << 40)
    assert (r["tier"] == 0).sum() == 49 and (r["tier"] == 1).sum() == 1


def test_program_larger_than_tier_blocks_the_prefix():
    # DESIGN R3: filling stops at the first program that does not fit
    iota = np.array([0.1, 0.2, 0.3, 0.4], np.float32)
    s = np.array([2, 50, 1, 1], np.int32)
    r = oracle.rank_partition(iota, s, None, 10, 10)
    assert r["tier"].tolist() == [0, 2, 2, 2] and r["bounds"].tolist() == [1, 1]
    r = oracle.rank_partition(iota, s, None, 10, 60)
    assert r["tier"].tolist() == [0, 1, 1, 1]


def test_zero_size_programs_take_the_tier_of_their_rank():
    iota = np.array([0.1, 0.2, 0.3, 0.4, 0.5], np.float32)
    s = np.array([5, 0, 5, 0, 5], np.int32)
    r = oracle.rank_partition(iota, s, None, 5, 5)
    assert r["tier"].tolist() == [0, 0, 1, 1, 2]


def test_bad_arguments_rejected():
    with pytest.raises(ValueError):
        oracle.rank_partition(np.zeros(2, np.float32), np.array([1, -1], np.int32), None, 1, 1)
    with pytest.raises(ValueError):
        oracle.rank_partition(np.zeros(2, np.float32), np.ones(2, np.int32), None, -1, 1)


def test_int64_accumulation():
    n = 4096
    s = np.full(n, 2 ** 31 - 1, np.int32)
    r = oracle.rank_partition(np.zeros(n, np.float32), s, None, 3000 * (2 ** 31 - 1), 10 ** 18)
    assert r["bounds"].tolist() == [3000, n] and r["used"][0] == 3000 * (2 ** 31 - 1)


# ---------------------------------------------------------------- movers
def _mk(rng, L, P, S, chunk):
    pool = rng.integers(0, 256, L * P * chunk, dtype=np.uint8)
    arena = rng.integers(0, 256, S * L * chunk, dtype=np.uint8)
    return pool, arena


def test_demote_matches_python_loops_and_fancy_index():
    rng = np.random.default_rng(7)
    L, P, S, chunk = 3, 11, 13, 32
    pool, arena = _mk(rng, L, P, S, chunk)
    g = rng.permutation(P)[:6].astype(np.int32)
    h = rng.permutation(S)[:6].astype(np.int32)
    want = arena.copy()
    for j in range(6):                        # byte-by-byte statement of SURVEY 8(c2)
        for l in range(L):
            for b in range(chunk):
                want[(h[j] * L + l) * chunk + b] = pool[(l * P + g[j]) * chunk + b]
    a1, a2 = arena.copy(), arena.copy()
    oracle.demote(L, chunk, pool, a1, g, h)
    oracle_np.demote(L, chunk, pool, a2, g, h)
    assert np.array_equal(a1, want) and np.array_equal(a2, want)
    # promote: mirror
    wantp = pool.copy()
    for j in range(6):
        for l in range(L):
            wantp[(l * P + g[j]) * chunk:(l * P + g[j] + 1) * chunk] = \
                arena[(h[j] * L + l) * chunk:(h[j] * L + l + 1) * chunk]
    p1, p2 = pool.copy(), pool.copy()
    oracle.promote(L, chunk, p1, arena, h, g)
    oracle_np.promote(L, chunk, p2, arena, h, g)
    assert np.array_equal(p1, wantp) and np.array_equal(p2, wantp)


def test_round_trip_returns_identical_pages_and_touches_nothing_else():
    # a promoted program "reload[s] the cache locally ... rather than recomputing"
    rng = np.random.default_rng(8)
    L, P, S, chunk = 4, 64, 40, 256
    pool, arena = _mk(rng, L, P, S, chunk)
    pool0, arena0 = pool.copy(), arena.copy()
    perm = rng.permutation(P)
    g, g2 = perm[:17].astype(np.int32), perm[17:34].astype(np.int32)
    h = rng.permutation(S)[:17].astype(np.int32)
    oracle.demote(L, chunk, pool, arena, g, h)
    assert np.array_equal(pool, pool0)                                   # source untouched
    av, av0 = arena.reshape(S, L, chunk), arena0.reshape(S, L, chunk)
    untouched = np.setdiff1d(np.arange(S), h)
    assert np.array_equal(av[untouched], av0[untouched])
    oracle.promote(L, chunk, pool, arena, h, g2)
    pv, pv0 = pool.reshape(L, P, chunk), pool0.reshape(L, P, chunk)
    assert np.array_equal(pv[:, g2], pv0[:, g])                          # identical logical pages
    other = np.setdiff1d(np.arange(P), g2)
    assert np.array_equal(pv[:, other], pv0[:, other])


def test_movers_reject_out_of_range_ids_and_accept_empty():
    pool, arena = np.zeros(2 * 4 * 8, np.uint8), np.zeros(3 * 2 * 8, np.uint8)
    with pytest.raises(ValueError):
        oracle.demote(2, 8, pool, arena, np.array([4], np.int32), np.array([0], np.int32))
    with pytest.raises(ValueError):
        oracle.promote(2, 8, pool, arena, np.array([3], np.int32), np.array([0], np.int32))
    oracle.demote(2, 8, pool, arena, np.zeros(0, np.int32), np.zeros(0, np.int32))
