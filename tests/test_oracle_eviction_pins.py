"""Pins of the typed-eviction-order oracle (NEXT-3): a hand-worked example, a lexsort
restatement, repeated selection of the minimum (no sort), and the paper's structural properties
(inactive first in both tiers, the busy/idle order reversed between them, LRU inside a type).
CPU only."""
import os

import numpy as np
import pytest

import oracle
from oracle import oracle_np

GOLD = os.path.join(os.path.dirname(__file__), "golden", "eviction_handworked.txt")


def _gold():
    d = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            d[k] = np.array(v, np.int64)
    return d


def rand_eviction_case(rng, n_pages, n_programs):
    owner = rng.integers(-1, n_programs, n_pages).astype(np.int32)
    ptier = rng.integers(0, 3, max(n_programs, 1)).astype(np.uint8)
    kind = rng.integers(0, 3)
    hi = [4, 1000, 2 ** 32][kind]
    last = rng.integers(0, hi, n_pages, dtype=np.uint64).astype(np.uint32)
    return owner, ptier, last


def test_hand_worked_example():
    g = _gold()
    for which, name in ((0, "gpu"), (1, "cpu")):
        for impl in (oracle.eviction_order, oracle_np.eviction_order):
            assert impl(which, g["owner"], g["program_tier"], g["last_access"]).tolist() == g[name].tolist()


@pytest.mark.parametrize("n_pages", [0, 1, 5, 64, 1000, 20000])
def test_c_oracle_equals_lexsort(n_pages):
    rng = np.random.default_rng(n_pages)
    for _ in range(6):
        case = rand_eviction_case(rng, n_pages, int(rng.integers(1, 50)))
        for which in (0, 1):
            assert np.array_equal(oracle.eviction_order(which, *case), oracle_np.eviction_order(which, *case))


def test_equals_repeatedly_evicting_the_best_victim():
    """No sort: pick, one at a time, the resident page with the lowest (type rank, last access,
    page id) -- what an engine evicting page by page under pressure would do."""
    rng = np.random.default_rng(3)
    for _ in range(30):
        owner, ptier, last = rand_eviction_case(rng, int(rng.integers(1, 40)), 6)
        for which in (0, 1):
            rank_of = {0: (2 if which == 0 else 1), 1: (1 if which == 0 else 2), 2: 0}   # by program tier
            left = [j for j in range(len(owner)) if owner[j] >= 0]
            seq = []
            while left:
                best = min(left, key=lambda j: (rank_of[int(ptier[owner[j]])], int(last[j]), j))
                seq.append(best); left.remove(best)
            assert oracle.eviction_order(which, owner, ptier, last).tolist() == seq


def test_structure_the_paper_states():
    rng = np.random.default_rng(8)
    owner, ptier, last = rand_eviction_case(rng, 3000, 40)
    label = np.where(owner >= 0, ptier[np.maximum(owner, 0)], 9)       # 0 busy, 1 idle, 2 inactive
    g, c = oracle.eviction_order(0, owner, ptier, last), oracle.eviction_order(1, owner, ptier, last)
    assert sorted(g.tolist()) == sorted(c.tolist()) == np.flatnonzero(owner >= 0).tolist()
    lg, lc = label[g], label[c]
    n_in, n_idle, n_busy = (label == 2).sum(), (label == 1).sum(), (label == 0).sum()
    assert (lg[:n_in] == 2).all() and (lc[:n_in] == 2).all()           # inactive first in both tiers
    assert (lg[n_in:n_in + n_idle] == 1).all() and (lg[n_in + n_idle:] == 0).all()    # GPU: idle, busy last
    assert (lc[n_in:n_in + n_busy] == 0).all() and (lc[n_in + n_busy:] == 1).all()    # CPU: busy, idle last
    for seq, lab in ((g, lg), (c, lc)):                                 # LRU inside every type
        for t in (0, 1, 2):
            assert (np.diff(last[seq[lab == t]].astype(np.int64)) >= 0).all()


def test_bad_arguments():
    with pytest.raises(ValueError):
        oracle.eviction_order(2, [0], [0], [0])
    with pytest.raises(ValueError):
        oracle.eviction_order(0, [5], [0], [0])           # owner past the program table
