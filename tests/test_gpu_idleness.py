"""Parity of mori_idleness_update / mori_idleness_eval (CUDA, through the C ABI) with the Eq. (1)
oracle: the float32 scores must be bit-identical (both sides sum in double in the same order,
divide once, round once); NaN only has to be NaN on both sides."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_00866_b200 import workload as W

pytestmark = pytest.mark.gpu


def _ctx(mori, n, k=0):
    pool = torch.zeros(2 * 4 * 8192, dtype=torch.uint8, device="cuda")
    return mori.Mori(2, 2, 64, 16, pool, max_programs=max(1, n), idleness_window=k)


def _dev(x, dt):
    return torch.from_numpy(np.ascontiguousarray(x, dtype=dt)).cuda()


def _update(m, prog, kind, r, a):
    m.mori_idleness_update(_dev(prog, np.int32), _dev(kind, np.uint8), _dev(r, np.float64), _dev(a, np.float64))


def _eval(m, n, open_r, open_a):
    out = torch.full((max(n, 1),), -1.0, dtype=torch.float32, device="cuda")
    m.mori_idleness_eval(n, None if open_r is None else _dev(open_r, np.float64),
                         None if open_a is None else _dev(open_a, np.float64), out)
    torch.cuda.synchronize()
    return out.cpu().numpy()[:n]


def assert_bits(got, want, tag=""):
    nan = np.isnan(want)
    assert np.array_equal(np.isnan(got), nan), tag
    assert np.array_equal(got[~nan].view(np.uint32), want[~nan].view(np.uint32)), tag


@pytest.mark.parametrize("n,k", [(1, 0), (7, 0), (300, 0), (4096, 0), (8192, 0), (50, 1), (50, 3), (50, 8)])
def test_random_event_streams_bit_exact(mori, n, k):
    m = _ctx(mori, n, k)
    t = oracle.IdlenessTracker(n, k or 5)
    rng = np.random.default_rng(n * 10 + k)
    assert_bits(_eval(m, n, None, None), t.eval(), "empty")          # nothing pushed: NaN everywhere
    for step in range(12):
        cnt = int(rng.integers(0, 3 * n + 2))                         # several events per program per call
        prog = rng.integers(0, n, cnt)
        kind = (rng.random(cnt) < 0.08).astype(np.uint8)
        r = rng.lognormal(1.4, 0.5, cnt); a = rng.lognormal(1.0, 1.5, cnt)
        a[rng.random(cnt) < 0.1] = 0.0
        t.update(prog, kind, r, a); _update(m, prog, kind, r, a)
        open_r = np.where(rng.random(n) < 0.5, rng.lognormal(1.0, 0.5, n), 0.0)
        open_a = np.where(rng.random(n) < 0.5, rng.lognormal(2.0, 1.5, n), 0.0)
        assert_bits(_eval(m, n, open_r, open_a), t.eval(open_r, open_a), (n, k, step))
        assert_bits(_eval(m, n, None, None), t.eval(), (n, k, step, "closed"))
    m.close()


@pytest.mark.parametrize("idx,scale,ticks", [(2, 64, 80), (4, 64, 40)])
def test_trace_ticks_feed_the_ranker_on_one_stream(mori, idx, scale, ticks):
    """Events of the synthetic agent trace -> device tracker -> iota -> mori_rank_partition on the
    same stream, never touching the host: scores bit-equal to the oracle (and to the trace
    generator's own), placement bit-equal to the oracle's."""
    cfg = W.get_config(idx, scale)
    n = cfg.n_programs
    m = _ctx(mori, n)
    tr = W.Trace(cfg, 866)
    t = oracle.IdlenessTracker(n)
    d = "cuda"
    iota_d = torch.empty(n, dtype=torch.float32, device=d)
    order = torch.empty(n, dtype=torch.int32, device=d); tier_d = torch.empty(n, dtype=torch.uint8, device=d)
    bounds = torch.empty(2, dtype=torch.int32, device=d); used = torch.empty(2, dtype=torch.int64, device=d)
    tier = np.full(n, 2, np.uint8)
    T = cfg.shape.page_tokens
    for e in range(ticks):
        iota_trace, tokens, _ = tr.advance(tier)
        prog, kind, r, a, open_r, open_a = tr.take_events()
        t.update(prog, kind, r, a)
        want_iota = t.eval(open_r, open_a)
        kv = ((tokens + T - 1) // T).astype(np.int32)
        if prog.size:
            _update(m, prog, kind, r, a)
        m.mori_idleness_eval(n, _dev(open_r, np.float64), _dev(open_a, np.float64), iota_d)
        m.mori_rank_partition(n, iota_d, _dev(kv, np.int32), None, cfg.cap_gpu_pages, cfg.cap_cpu_pages,
                              order, tier_d, bounds, used)
        torch.cuda.synchronize()
        assert_bits(iota_d.cpu().numpy(), want_iota, e)
        assert np.array_equal(want_iota.view(np.uint32), iota_trace.view(np.uint32))
        want = oracle.rank_partition(want_iota, kv, None, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        assert np.array_equal(order.cpu().numpy(), want["order"]) and np.array_equal(tier_d.cpu().numpy(), want["tier"])
        tier = want["tier"]
    m.close()


def test_argument_errors(mori):
    m = _ctx(mori, 8)
    z = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(mori.MoriError):
        m.mori_idleness_eval(9, None, None, z)
    with pytest.raises(mori.MoriError):
        m.mori_idleness_eval(4, None, None, None)
    m.mori_idleness_eval(0, None, None, None)
    m.close()
    with pytest.raises(mori.MoriError):
        _ctx(mori, 8, k=65)
