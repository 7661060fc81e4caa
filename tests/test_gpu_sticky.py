"""Parity of mori_sticky_rebalance (CUDA, through the C ABI) with the CPU oracle of the paper's
section 4.3.1: bit-exact tiers, lazy flags, used pages and all lists."""
import numpy as np
import pytest
import torch

import oracle
from test_oracle_sticky_pins import rand_sticky_case, _gold

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(mori):
    pool = torch.zeros(2 * 4 * 8192, dtype=torch.uint8, device="cuda")
    m = mori.Mori(2, 2, 64, 16, pool)
    yield m
    m.close()


def gpu_sticky(m, iota, s, prev, flags, cg, cc):
    n, d = len(s), "cuda"
    t = [torch.from_numpy(np.ascontiguousarray(x, dtype=dt)).to(d)
         for x, dt in ((iota, np.float32), (s, np.int32), (prev, np.uint8), (flags, np.uint8))]
    tier = torch.full((max(n, 1),), 9, dtype=torch.uint8, device=d)
    lazy = torch.full((max(n, 1),), 9, dtype=torch.uint8, device=d)
    used = torch.full((2,), -7, dtype=torch.int64, device=d)
    lists = torch.full((5 * max(n, 1),), -7, dtype=torch.int32, device=d)
    counts = torch.full((5,), -7, dtype=torch.int32, device=d)
    m.mori_sticky_rebalance(n, t[0], t[1], t[2], t[3], cg, cc, tier, lazy, used, lists, counts)
    torch.cuda.synchronize()
    c = counts.cpu().numpy()
    l2 = lists.cpu().numpy()[:5 * n].reshape(5, n) if n else np.zeros((5, 0), np.int32)
    return dict(tier=tier.cpu().numpy()[:n], lazy=lazy.cpu().numpy()[:n], used=used.cpu().numpy(),
                lists=[l2[k, :c[k]] for k in range(5)])


def assert_same(a, b, tag=""):
    for k in ("tier", "lazy", "used"):
        assert np.array_equal(a[k], b[k]), (tag, k)
    for k in range(5):
        assert np.array_equal(a["lists"][k], b["lists"][k]), (tag, "list", k)


def test_hand_worked_ticks(ctx):
    g = _gold()
    iota = np.array(g["iota"], np.float32)
    s, prev, fl = (np.array(g[k], np.int64) for k in ("pages", "prev_tier", "flags"))
    for suffix in ("", "2", "3"):
        cg, cc = map(int, g["cap" + suffix])
        got = gpu_sticky(ctx, iota, s, prev, fl, cg, cc)
        assert got["tier"].tolist() == list(map(int, g["tier" + suffix]))
        assert got["used"].tolist() == list(map(int, g["used" + suffix]))
        assert_same(got, oracle.sticky_rebalance(iota, s, prev, fl, cg, cc), suffix)


@pytest.mark.parametrize("n", [0, 1, 2, 7, 31, 32, 33, 64, 256, 1000, 1024, 1025, 2048, 3000, 4096,
                               4097, 8191, 8192])
def test_random_ticks_bit_exact(ctx, n):
    rng = np.random.default_rng(700 + n)
    for rep in range(8):
        case = rand_sticky_case(rng, n, tight=rep % 2 == 0)
        assert_same(gpu_sticky(ctx, *case), oracle.sticky_rebalance(*case), (n, rep))


def test_cpu_full_forces_the_per_victim_walk(ctx):
    """CPU queue nearly full: some victims fit, later smaller ones still do (the sequential
    'CPU if it fits, else Waiting' of P:L206), on a large n."""
    rng = np.random.default_rng(5)
    n = 6000
    iota = rng.random(n).astype(np.float32)
    s = rng.integers(1, 50, n).astype(np.int32)
    prev = np.zeros(n, np.uint8)
    prev[rng.random(n) < 0.3] = 1
    flags = rng.integers(0, 8, n).astype(np.uint8)
    cc = int(s[prev == 1].sum()) + 500
    cg = int(s[prev == 0].sum()) // 3
    got = gpu_sticky(ctx, iota, s, prev, flags, cg, cc)
    want = oracle.sticky_rebalance(iota, s, prev, flags, cg, cc)
    assert want["lists"][0].size > 5 and want["lists"][2].size > 100
    assert_same(got, want)


def test_argument_errors(ctx, mori):
    z = torch.zeros(8, dtype=torch.uint8, device="cuda")
    with pytest.raises(mori.MoriError) as e:
        ctx.mori_sticky_rebalance(9000, z, z, z, z, 1, 1, z, z, z, z, z)
    assert e.value.code == mori.ERR_INVALID_ARG
    with pytest.raises(mori.MoriError):
        ctx.mori_sticky_rebalance(4, z, z, z, z, -1, 1, z, z, z, z, z)
    with pytest.raises(mori.MoriError):
        ctx.mori_sticky_rebalance(4, None, z, z, z, 1, 1, z, z, z, z, z)
