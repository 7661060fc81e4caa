"""Parity of mori_rank_partition (CUDA, through the C ABI) with the CPU oracle: bit-exact on
order, tier, bounds, used pages and all five lists."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_00866_b200 import workload as W
from test_oracle_pins import _rand_case

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(mori):
    pool = torch.zeros(2 * 4 * 8192, dtype=torch.uint8, device="cuda")
    m = mori.Mori(2, 2, 64, 16, pool)          # no arena: rank/partition only
    yield m
    m.close()


def gpu_rank(m, iota, s, prev, cg, cc):
    n = len(iota)
    d = "cuda"
    t_i = torch.from_numpy(np.asarray(iota, np.float32)).to(d)
    t_s = torch.from_numpy(np.asarray(s, np.int32)).to(d)
    t_p = None if prev is None else torch.from_numpy(np.asarray(prev, np.uint8)).to(d)
    order = torch.full((max(n, 1),), -7, dtype=torch.int32, device=d)
    tier = torch.full((max(n, 1),), 9, dtype=torch.uint8, device=d)
    bounds = torch.full((2,), -7, dtype=torch.int32, device=d)
    used = torch.full((2,), -7, dtype=torch.int64, device=d)
    lists = torch.full((5, max(n, 1)), -7, dtype=torch.int32, device=d)
    counts = torch.full((5,), -7, dtype=torch.int32, device=d)
    m.mori_rank_partition(n, t_i, t_s, t_p, cg, cc, order, tier, bounds, used,
                          lists if prev is not None else None, counts if prev is not None else None)
    torch.cuda.synchronize()
    out = dict(order=order.cpu().numpy()[:n], tier=tier.cpu().numpy()[:n], bounds=bounds.cpu().numpy(),
               used=used.cpu().numpy())
    if prev is not None:
        c = counts.cpu().numpy()
        l2 = lists.cpu().numpy().reshape(-1)[:5 * n].reshape(5, n) if n else np.zeros((5, 0), np.int32)
        out["lists"] = [l2[k, :c[k]] for k in range(5)]
    return out


def assert_same(a, b, tag=""):
    for k in ("order", "tier", "bounds", "used"):
        assert np.array_equal(a[k], b[k]), (tag, k, a[k][:10], b[k][:10])
    if "lists" in b:
        for k in range(5):
            assert np.array_equal(a["lists"][k], b["lists"][k]), (tag, "list", k)


@pytest.mark.parametrize("n", [0, 1, 2, 7, 8, 31, 32, 33, 64, 128, 256, 1000, 1024, 1025, 2048,
                               3000, 4096, 4097, 8191, 8192])
def test_random_cases_bit_exact(ctx, n):
    rng = np.random.default_rng(100 + n)
    for rep in range(6):
        iota, s, prev, cg, cc = _rand_case(rng, n)
        want = oracle.rank_partition(iota, s, prev, cg, cc)
        got = gpu_rank(ctx, iota, s, prev, cg, cc)
        assert_same(got, want, (n, rep))
    iota, s, prev, cg, cc = _rand_case(rng, n)
    assert_same(gpu_rank(ctx, iota, s, None, cg, cc), oracle.rank_partition(iota, s, None, cg, cc))


def test_degenerate_inputs(ctx):
    n = 4096
    ones = np.ones(n, np.int32)
    cases = [
        (np.zeros(n, np.float32), ones, 100, 200),                        # all ties -> identity order
        (np.linspace(1, 0, n).astype(np.float32), ones, 100, 200),        # reversal
        (np.full(n, np.nan, np.float32), ones, 5, 5),                     # all NaN
        (np.where(np.arange(n) % 2, 0.0, -0.0).astype(np.float32), ones, 7, 9),   # signed zeros tie
        (np.random.default_rng(1).random(n).astype(np.float32), ones * 0, 0, 0),  # zero sizes, zero caps
        (np.random.default_rng(2).random(n).astype(np.float32), ones * (2 ** 31 - 1),
         3000 * (2 ** 31 - 1), 10 ** 18),                                 # int64 accumulation
        (np.random.default_rng(3).random(n).astype(np.float32), ones, 0, n),
        (np.random.default_rng(4).random(n).astype(np.float32), ones, n, 0),
        (np.random.default_rng(5).random(n).astype(np.float32), ones, 2 ** 62, 2 ** 62),
    ]
    prev = np.random.default_rng(9).integers(0, 4, n).astype(np.uint8)     # value 3 -> WAIT
    for i, (iota, s, cg, cc) in enumerate(cases):
        assert_same(gpu_rank(ctx, iota, s, prev, cg, cc), oracle.rank_partition(iota, s, prev, cg, cc), i)


def test_program_larger_than_tier(ctx):
    iota = np.array([0.1, 0.2, 0.3, 0.4], np.float32)
    s = np.array([2, 50, 1, 1], np.int32)
    prev = np.zeros(4, np.uint8)
    for cg, cc in [(10, 10), (10, 60), (1, 1)]:
        assert_same(gpu_rank(ctx, iota, s, prev, cg, cc), oracle.rank_partition(iota, s, prev, cg, cc))


def test_argument_errors(ctx, mori):
    d = "cuda"
    z = torch.zeros(8, dtype=torch.int32, device=d)
    f = torch.zeros(8, dtype=torch.float32, device=d)
    u = torch.zeros(8, dtype=torch.uint8, device=d)
    b = torch.zeros(2, dtype=torch.int32, device=d)
    us = torch.zeros(2, dtype=torch.int64, device=d)
    for kw in [dict(n=-1), dict(n=8193), dict(cg=-1), dict(cc=-1)]:
        with pytest.raises(mori.MoriError) as e:
            ctx.mori_rank_partition(kw.get("n", 8), f, z, None, kw.get("cg", 1), kw.get("cc", 1), z, u, b, us)
        assert e.value.code == mori.ERR_INVALID_ARG
    with pytest.raises(mori.MoriError):
        ctx.mori_rank_partition(8, f, z, u, 1, 1, z, u, b, us, None, None)   # prev_tier without lists


# BASELINE.json's configs as written: full size, full epoch counts (20 / 200 / 200 x 3 / 100 / 500);
# cfg 3 is three runs, the busy:idle ratio swept 1:3, 1:1, 3:1 (f_busy 0.25 / 0.5 / 0.75) "so the
# partition boundary moves".
@pytest.mark.parametrize("idx,f_busy,epochs", [(1, None, 20), (2, None, 200), (3, 0.25, 200), (3, 0.5, 200),
                                               (3, 0.75, 200), (4, None, 100), (5, None, 500)])
def test_config_traces_full_size_placement(ctx, idx, f_busy, epochs):
    """Placement on the configs' own traces at FULL size (placement needs no pools): every epoch
    bit-exact; the sim advances on the oracle's placement.  Seed 866 runs every epoch BASELINE.json
    asks for, seeds 867 / 868 the first 20."""
    cfg = W.get_config(idx, 1, f_busy)
    assert cfg.epochs == epochs
    b_gpu_seen = set()
    for seed in (866, 867, 868):
        sim = W.Sim(cfg, seed)
        for e in range(epochs if seed == 866 else min(epochs, 20)):
            plan = sim.begin_epoch()
            want = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
            got = gpu_rank(ctx, plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
            assert_same(got, want, (cfg.name, seed, e))
            if idx == 1:
                b = oracle.bruteforce_partition(plan.iota, plan.kv_pages, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
                assert np.array_equal(b["tier"], got["tier"])
            b_gpu_seen.add(int(got["bounds"][0]))
            sim.apply_placement(want["tier"], want["lists"])
            sim.end_epoch()
    if idx in (2, 3, 4, 5):
        assert len(b_gpu_seen) > 3, "the partition boundary never moved"
