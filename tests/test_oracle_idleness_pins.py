"""Pins of the Eq. (1) oracle (NEXT-2): the closed forms of tests/golden/eq1_examples.txt,
window slide, outlier dilution and responsiveness as the paper describes them, exact rational
arithmetic on small integers, and bit-equality with the trace generator's own (numpy) statement
of the same window.  CPU only."""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2606_00866_b200 import workload as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "eq1_examples.txt")


def _push(t, p, pairs):
    for r, a in pairs:
        t.update([p], [0], [r], [a])


def test_golden_closed_forms():
    rows = [l for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) >= 5
    for line in rows:
        r, a, want = [x.split() for x in line.split("|")]
        t = oracle.IdlenessTracker(1)
        _push(t, 0, zip(map(float, r), map(float, a)))
        assert t.eval()[0] == np.float32(float(want[0]))


def test_exact_rational_value_and_single_rounding():
    rng = np.random.default_rng(1)
    for _ in range(200):
        k = int(rng.integers(1, 6))
        r = rng.integers(0, 1000, k); a = rng.integers(0, 1000, k)
        if r.sum() + a.sum() == 0:
            continue
        t = oracle.IdlenessTracker(1)
        _push(t, 0, zip(r.astype(float), a.astype(float)))
        exact = Fraction(int(a.sum()), int(r.sum() + a.sum()))
        # integer sums are exact in double; one division (correctly rounded) then one rounding to f32
        assert t.eval()[0] == np.float32(float(exact))


def test_window_slides_after_k_cycles_and_reset_clears():
    t = oracle.IdlenessTracker(2)
    _push(t, 0, [(1, 99)] + [(1, 1)] * 5)          # the long call is pushed out by 5 short ones
    assert t.eval()[0] == np.float32(0.5)
    _push(t, 1, [(1, 99)] + [(1, 1)] * 4)          # still inside the window of 5
    assert t.eval()[1] == np.float32(103 / 108)
    t.update([1], [1], [0.0], [0.0])               # slot reused by a new program
    assert np.isnan(t.eval()[1]) and t.eval()[0] == np.float32(0.5)
    _push(t, 1, [(3, 1)])
    assert t.eval()[1] == np.float32(0.25)


def test_open_cycle_is_the_newest_of_the_k_and_dominates_as_it_grows():
    """'the ongoing tool call's elapsed time keeps increasing and soon dominates'."""
    t = oracle.IdlenessTracker(1)
    _push(t, 0, [(4, 1)] * 5)                      # busy phase: iota = 0.2
    assert t.eval()[0] == np.float32(0.2)
    prev = -1.0
    for elapsed in (0.5, 5, 50, 500):
        v = t.eval([4.0], [elapsed])[0]            # open cycle: 4 s reasoning done, tool call running
        want = (4 * 1 + elapsed) / (4 * 4 + 4 + 4 * 1 + elapsed)   # 4 completed + the open one
        assert v == np.float32(want) and v > prev
        prev = v
    assert prev > 0.95
    assert t.eval([0.0], [0.0])[0] == np.float32(0.2)              # no elapsed time: not a cycle


def test_outlier_dilution():
    """one unexpectedly long call among short ones does not flip a busy program ..."""
    t = oracle.IdlenessTracker(2)
    _push(t, 0, [(4, 1)] * 4 + [(4, 10)])
    assert t.eval()[0] == np.float32(14 / 34) and t.eval()[0] < 0.5
    _push(t, 1, [(4, 60)] * 5)                     # ... sustained long calls do
    assert t.eval()[1] > 0.9


@pytest.mark.parametrize("idx,scale,ticks", [(1, 1, 60), (2, 64, 120), (3, 64, 60)])
def test_bit_equal_to_the_trace_generators_own_window(idx, scale, ticks):
    """workload.Trace computes iota with numpy slices of its own per-program history lists; the
    oracle is fed only the event stream a router would see.  Two statements, same bits."""
    cfg = W.get_config(idx, scale)
    tr = W.Trace(cfg, 866)
    t = oracle.IdlenessTracker(cfg.n_programs)
    rng = np.random.default_rng(3)
    tier = np.zeros(cfg.n_programs, np.uint8)
    for e in range(ticks):
        if e % 5 == 2:                              # gate a random half: gated time must not count
            tier = (rng.random(cfg.n_programs) < 0.5).astype(np.uint8) * 2
        iota, _, _ = tr.advance(tier)
        prog, kind, r, a, open_r, open_a = tr.take_events()
        t.update(prog, kind, r, a)
        got = t.eval(open_r, open_a)
        assert np.array_equal(got.view(np.uint32), iota.view(np.uint32)), e


def test_bad_program_index_rejected():
    t = oracle.IdlenessTracker(2)
    with pytest.raises(ValueError):
        t.update([2], [0], [1.0], [1.0])
