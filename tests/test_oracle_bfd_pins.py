"""Pins of the Best-Fit-Decreasing oracle (NEXT-4(i)): a hand-worked packing, a numpy
restatement, the single-replica special case (plain first-fit-decreasing into one bin), and the
properties the rule implies.  CPU only."""
import os

import numpy as np
import pytest

import oracle
from oracle import oracle_np

GOLD = os.path.join(os.path.dirname(__file__), "golden", "bfd_handworked.txt")


def _gold():
    d = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            d[k] = np.array(v, np.float64)
    return d


def rand_bfd_case(rng, m, R):
    size = rng.integers(0, 40, m).astype(np.int32)
    if m and rng.random() < 0.5:
        size[:] = rng.choice([3, 5, 8], m)                 # many equal sizes: the tie rules matter
    iota = np.round(rng.random(m) * 8).astype(np.float32) / 8
    flags = (2 | (rng.integers(0, 2, m) * 4)).astype(np.uint8)
    free = rng.integers(0, max(2, int(size.sum()) // max(1, R) + 10), R).astype(np.int64)
    return size, iota, flags, free


def test_hand_worked_packing():
    g = _gold()
    for impl in (oracle.bfd_assign, oracle_np.bfd_assign):
        rep, free = impl(g["size"], g["iota"].astype(np.float32), g["flags"].astype(np.uint8), g["free"])
        assert rep.tolist() == g["replica"].astype(int).tolist()
        assert free.tolist() == g["free_out"].astype(int).tolist()


@pytest.mark.parametrize("m,R", [(0, 1), (1, 1), (5, 3), (40, 8), (300, 2), (2000, 32)])
def test_c_oracle_equals_numpy_restatement(m, R):
    rng = np.random.default_rng(m * 100 + R)
    for _ in range(10):
        case = rand_bfd_case(rng, m, R)
        a, b = oracle.bfd_assign(*case), oracle_np.bfd_assign(*case)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_single_replica_is_first_fit_decreasing_into_one_bin():
    rng = np.random.default_rng(5)
    for _ in range(50):
        size, iota, flags, free = rand_bfd_case(rng, int(rng.integers(1, 30)), 1)
        size = np.unique(size)                                        # distinct sizes: order is by size alone
        iota, flags = iota[:size.size], flags[:size.size]
        rep, left = oracle.bfd_assign(size, iota, flags, free)
        cap, want = int(free[0]), {}
        for i in np.argsort(-size):
            want[i] = 0 if size[i] <= cap else -1
            cap -= size[i] if want[i] == 0 else 0
        assert rep.tolist() == [want[i] for i in range(size.size)] and left[0] == cap


def test_properties():
    rng = np.random.default_rng(6)
    for _ in range(200):
        m, R = int(rng.integers(0, 60)), int(rng.integers(1, 9))
        size, iota, flags, free = rand_bfd_case(rng, m, R)
        rep, left = oracle.bfd_assign(size, iota, flags, free)
        assert ((rep >= -1) & (rep < R)).all() and (left >= 0).all()
        for r in range(R):                                            # conservation per replica
            assert left[r] == free[r] - size[rep == r].sum()
        # a candidate left in Waiting is larger than everything that was still free when its turn
        # came; free space only shrinks, so it is larger than every replica's final free space too
        if (rep == -1).any():
            assert size[rep == -1].min() > left.max()
        # among equal sizes, a returning program is never left behind while a new one is admitted
        for s in np.unique(size):
            eq = size == s
            new = (flags & 4) != 0
            if (eq & ~new & (rep == -1)).any():
                assert not (eq & new & (rep >= 0)).any()


def test_bad_arguments():
    with pytest.raises(ValueError):
        oracle.bfd_assign([1], [0.1], [2], [-1])
    with pytest.raises(ValueError):
        oracle.bfd_assign([-1], [0.1], [2], [5])
