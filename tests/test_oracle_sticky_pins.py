"""Pins of the sticky, status-aware tier management oracle (NEXT-1; paper section 4.3.1):
a hand-worked tick, a second independent statement (sorts + prefix sums vs one-at-a-time
selection), reduction to the already pinned rank/partition, invariants, and a brute force of
the demotion step.  CPU only."""
import itertools
import os

import numpy as np
import pytest

import oracle
from oracle import oracle_np

GOLD = os.path.join(os.path.dirname(__file__), "golden", "sticky_handworked.txt")
ACTING, READY, NEW = 1, 2, 4


def _gold():
    d = {}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        d[k] = v
    return d


def _same(a, b):
    for k in ("tier", "lazy", "used"):
        assert np.array_equal(a[k], b[k]), k
    for k in range(5):
        assert np.array_equal(a["lists"][k], b["lists"][k]), ("list", k)


def test_hand_worked_ticks():
    g = _gold()
    iota = np.array(g["iota"], np.float32)
    s, prev, fl = (np.array(g[k], np.int64) for k in ("pages", "prev_tier", "flags"))
    for suffix, lists in (("", dict(demote=0, promote=1, drop=2, admit=3)),
                          ("2", {}), ("3", dict(promote3=1, admit3=3))):
        cg, cc = map(int, g["cap" + suffix])
        for impl in (oracle.sticky_rebalance, oracle_np.sticky_rebalance):
            r = impl(iota, s, prev, fl, cg, cc)
            assert r["tier"].tolist() == list(map(int, g["tier" + suffix]))
            assert r["used"].tolist() == list(map(int, g["used" + suffix]))
            if suffix == "":
                assert r["lazy"].tolist() == list(map(int, g["lazy"]))
            want = {0: [], 1: [], 2: [], 3: [], 4: []}
            for name, row in lists.items():
                want[row] = list(map(int, g[name]))
            for k in range(5):
                assert r["lists"][k].tolist() == want[k], (suffix, k)


def rand_sticky_case(rng, n, tight=True):
    kind = rng.integers(0, 4)
    if kind == 0:
        iota = rng.random(n).astype(np.float32)
    elif kind == 1:
        iota = rng.choice(np.array([0.0, -0.0, 0.25, 0.5, 1.0, np.inf, -np.inf, np.nan], np.float32), n)
    elif kind == 2:
        iota = rng.lognormal(0, 1, n).astype(np.float32)
    else:
        iota = np.round(rng.random(n) * 4).astype(np.float32) / 4
    s = rng.integers(0, 9 if tight else 600, n).astype(np.int32)
    prev = rng.integers(0, 3, n).astype(np.uint8)
    flags = rng.integers(0, 8, n).astype(np.uint8)
    cpu_now = int(s[prev == 1].sum())
    gpu_now = int(s[prev == 0].sum())
    cap_cpu = cpu_now + int(rng.integers(0, max(2, int(s.sum()) // 3 + 1)))
    cap_gpu = int(rng.integers(0, max(2, 2 * gpu_now + 8)))
    return iota, s, prev, flags, cap_gpu, cap_cpu


@pytest.mark.parametrize("n", [0, 1, 2, 5, 17, 64, 300, 1500])
def test_c_oracle_equals_sort_and_scan_restatement(n):
    rng = np.random.default_rng(4000 + n)
    for rep in range(40 if n <= 64 else 8):
        case = rand_sticky_case(rng, n, tight=rep % 2 == 0)
        _same(oracle.sticky_rebalance(*case), oracle_np.sticky_rebalance(*case))


def test_reduces_to_rank_partition_when_everything_is_acting_on_gpu():
    """All programs on GPU, all Acting, unlimited CPU, nobody ready: demoting the most idle until
    the rest fits leaves exactly the longest busiest-first prefix that fits = the GPU tier of the
    (separately pinned) rank/partition, and the victims come out most idle first."""
    rng = np.random.default_rng(9)
    for n in (1, 7, 50, 400):
        for _ in range(10):
            iota = rng.random(n).astype(np.float32)
            iota[rng.integers(0, n, n // 4)] = 0.5                      # ties
            s = rng.integers(0, 20, n).astype(np.int32)
            cap = int(rng.integers(0, int(s.sum()) + 2))
            st = oracle.sticky_rebalance(iota, s, np.zeros(n, np.uint8), np.full(n, ACTING, np.uint8), cap, 1 << 40)
            rp = oracle.rank_partition(iota, s, np.zeros(n, np.uint8), cap, 1 << 40)
            b = int(rp["bounds"][0])
            # zero-size programs just past the cut fit the prefix but are still victims of the
            # one-at-a-time loop only while usage exceeds the cap: compare page totals and sets
            assert st["used"][0] == rp["used"][0]
            kept = set(np.flatnonzero(st["tier"] == 0).tolist())
            assert set(rp["order"][:b].tolist()) <= kept
            assert all(s[p] == 0 for p in kept - set(rp["order"][:b].tolist()))
            v = st["lists"][0].tolist()
            assert v == rp["order"][::-1][:len(v)].tolist()
            assert not st["lazy"].any() and st["lists"][2].size == 0


def _brute_demotion(iota, s, flags, gpu_set, cap):
    """Every subset of GPU programs to KEEP that fits and is closed under the victim priority
    (a kept program is never a better victim than a demoted one); the paper's loop demotes as few
    as possible in that order -> the largest such subset."""
    def worse_victim(a, b):          # a is demoted after b
        aa, ab = bool(flags[a] & ACTING), bool(flags[b] & ACTING)
        if aa != ab:
            return ab
        ka, kb = oracle_np.sort_key(np.array([iota[a]]))[0][0], oracle_np.sort_key(np.array([iota[b]]))[0][0]
        na, nb = np.isnan(iota[a]), np.isnan(iota[b])
        if na != nb:
            return nb
        if not na and ka != kb:
            return ka < kb
        return a < b
    best = None
    for r in range(len(gpu_set), -1, -1):
        for keep in itertools.combinations(gpu_set, r):
            if sum(int(s[p]) for p in keep) > cap:
                continue
            out = [p for p in gpu_set if p not in keep]
            if all(worse_victim(k, o) for k in keep for o in out):
                best = set(keep)
                break
        if best is not None:
            break
    return best


def test_demotion_is_the_minimal_victim_prefix_brute_force():
    rng = np.random.default_rng(77)
    for _ in range(150):
        n = int(rng.integers(1, 9))
        iota, s, prev, flags, cg, cc = rand_sticky_case(rng, n)
        s = np.maximum(s, 1)                                      # positive sizes: unique minimum
        prev[:] = 0
        flags &= ~np.uint8(READY)
        r = oracle.sticky_rebalance(iota, s, prev, flags, cg, 1 << 40)
        kept = set(np.flatnonzero(r["tier"] == 0).tolist())
        assert kept == _brute_demotion(iota, s, flags, list(range(n)), cg)


def check_sticky_invariants(case, r):
    iota, s, prev, flags, cg, cc = case
    n = len(s)
    prev = np.where(np.asarray(prev) > 2, 2, prev)
    tier, lists = r["tier"], r["lists"]
    s64 = np.asarray(s, np.int64)
    assert r["used"][0] == s64[tier == 0].sum() and r["used"][1] == s64[tier == 1].sum()
    assert r["used"][1] <= cc
    gpu_before = s64[prev == 0].sum()
    demoted = np.concatenate([lists[0], lists[2]])
    if gpu_before <= cg:
        assert demoted.size == 0                                   # sticky: no overflow, no demotion
    else:
        assert r["used"][0] <= cg or (tier == 0).sum() == 0 or s64[(tier == 0) & (prev == 0)].sum() <= cg
    moved = set(np.flatnonzero(tier != prev).tolist())
    assert moved == set(np.concatenate(lists[:4]).tolist())        # only listed programs change tier
    assert len(moved) == sum(len(x) for x in lists[:4])            # lists are disjoint
    assert all(prev[p] == 0 and tier[p] == 1 for p in lists[0])
    assert all(prev[p] == 1 and tier[p] == 0 and flags[p] & READY for p in lists[1])
    assert all(prev[p] == 0 and tier[p] == 2 for p in lists[2])
    assert all(prev[p] == 2 and tier[p] == 0 and flags[p] & READY for p in lists[3])
    assert lists[4].size == 0
    # Reasoning victims only once every Acting GPU program is gone; they are the lazy ones
    lazy = set(np.flatnonzero(r["lazy"]).tolist())
    assert lazy == {int(p) for p in demoted if not flags[p] & ACTING}
    if lazy:
        assert not any(tier[p] == 0 and prev[p] == 0 and flags[p] & ACTING for p in range(n))
    # promotions never overflow the GPU
    if lists[1].size + lists[3].size:
        assert r["used"][0] <= cg


def test_invariants_on_random_ticks():
    rng = np.random.default_rng(31)
    for _ in range(400):
        n = int(rng.integers(0, 40))
        case = rand_sticky_case(rng, n)
        check_sticky_invariants(case, oracle.sticky_rebalance(*case))


def test_bad_arguments_are_rejected():
    with pytest.raises(ValueError):
        oracle.sticky_rebalance([0.1], [5], [1], [0], 10, 4)        # CPU queue already over capacity
    with pytest.raises(ValueError):
        oracle.sticky_rebalance([0.1], [-1], [0], [0], 10, 4)
    with pytest.raises(ValueError):
        oracle.sticky_rebalance([0.1], [1], [0], [0], -1, 4)
