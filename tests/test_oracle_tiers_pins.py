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
