"""Parity of mori_rank_partition_tiers (CUDA, through the C ABI) with the T-capacity partition
oracle: bit-exact order, tier, bounds and used pages."""
import numpy as np
import pytest
import torch

import oracle
from test_oracle_pins import _rand_case

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(mori):
    pool = torch.zeros(2 * 4 * 8192, dtype=torch.uint8, device="cuda")
    m = mori.Mori(2, 2, 64, 16, pool)
    yield m
    m.close()


def gpu_tiers(m, iota, s, caps, prev=None):
    n, T, d = len(iota), len(caps), "cuda"
    order = torch.full((max(n, 1),), -7, dtype=torch.int32, device=d)
    tier = torch.full((max(n, 1),), 99, dtype=torch.uint8, device=d)
    bounds = torch.full((T,), -7, dtype=torch.int32, device=d)
    used = torch.full((T,), -7, dtype=torch.int64, device=d)
    t_prev = None if prev is None else torch.from_numpy(np.asarray(prev, np.uint8)).to(d)
    moves = torch.full((2 * max(n, 1),), -7, dtype=torch.int32, device=d)
    counts = torch.full((2,), -7, dtype=torch.int32, device=d)
    m.mori_rank_partition_tiers(n, torch.from_numpy(np.asarray(iota, np.float32)).to(d),
                                torch.from_numpy(np.asarray(s, np.int32)).to(d), caps, order, tier, bounds, used,
                                prev_tier=t_prev, moves=moves if prev is not None else None,
                                move_counts=counts if prev is not None else None)
    torch.cuda.synchronize()
    out = dict(order=order.cpu().numpy()[:n], tier=tier.cpu().numpy()[:n], bounds=bounds.cpu().numpy(),
               used=used.cpu().numpy())
    if prev is not None:
        c, mv = counts.cpu().numpy(), moves.cpu().numpy()
        out["moves"] = [mv[k * n:k * n + c[k]] for k in range(2)]
    return out


@pytest.mark.parametrize("n", [0, 1, 2, 31, 33, 64, 1000, 1024, 1025, 2048, 4096, 4097, 8192])
def test_random_cases_bit_exact(ctx, n):
    rng = np.random.default_rng(300 + n)
    for rep in range(6):
        iota, s, prev, cg, cc = _rand_case(rng, n)
        T = int(rng.integers(1, 9))
        caps = rng.integers(0, max(2, int(np.sum(s)) // max(1, T - 1) + 2), T)
        if rep == 0:
            caps[:] = 0
        pv = rng.integers(0, T + 2, n).astype(np.uint8) if rep % 2 else None
        got, want = gpu_tiers(ctx, iota, s, caps, pv), oracle.rank_partition_tiers(iota, s, caps, pv)
        for k in ("order", "tier", "bounds", "used"):
            assert np.array_equal(got[k], want[k]), (n, rep, k)
        if pv is not None:
            for k in range(2):
                assert np.array_equal(got["moves"][k], want["moves"][k]), (n, rep, "moves", k)


def test_two_tiers_equals_mori_rank_partition_on_a_config_trace(ctx, mori):
    from paper_2606_00866_b200 import workload as W
    cfg = W.get_config(5)
    tr = W.Trace(cfg, 866)
    T = cfg.shape.page_tokens
    for e in range(5):
        iota, tokens, _ = tr.advance(np.zeros(cfg.n_programs, np.uint8))
        kv = ((tokens + T - 1) // T).astype(np.int32)
        got = gpu_tiers(ctx, iota, kv, [cfg.cap_gpu_pages, cfg.cap_cpu_pages])
        want = oracle.rank_partition(iota, kv, None, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        for k in ("order", "tier", "bounds", "used"):
            assert np.array_equal(got[k], want[k]), (e, k)


def test_argument_errors(ctx, mori):
    z = torch.zeros(8, dtype=torch.int32, device="cuda")
    for caps in ([], [1] * 9, [3, -1]):
        with pytest.raises(mori.MoriError):
            ctx.mori_rank_partition_tiers(4, z, z, caps, z, z, z, z)


@pytest.mark.parametrize("idx,scale,mid_frac,epochs,slack_div", [(2, 128, 0.5, 30, 2), (3, 128, 0.4, 20, 2),
                                                                   (2, 128, 0.35, 32, 0)])
def test_three_tier_epochs_all_three_pools_byte_exact(mori, idx, scale, mid_frac, epochs, slack_div):
    """A whole epoch across three pools ("a second idleness threshold ... an intermediate
    tier"): mori_rank_partition_tiers decides (tiers and both move lists bit-exact vs the oracle),
    mori_demote / mori_promote of the three pair-contexts move the bytes (pool <-> device-resident
    middle arena, pool <-> pinned host arena, middle <-> host), and after every epoch the GPU pool,
    the middle arena and the host arena equal the oracle's three mirrors byte for byte."""
    from paper_2606_00866_b200 import workload as W
    from paper_2606_00866_b200.harness import TierRunner
    from test_oracle_tiers_pins import oracle_apply_moves
    cfg = W.get_config(idx, scale)
    sh = cfg.shape
    seed = 866
    mid_ids = int(cfg.gpu_pool_pages * mid_frac)
    pool_ids = [cfg.gpu_pool_pages, mid_ids, cfg.cpu_pool_pages]
    # slack_div = 0: the ranker is given every middle slot, so the planner must split epochs into
    # phases separated by joins (an id freed in a phase is not reused before the next join)
    slack = cfg.max_program_pages // slack_div if slack_div else 0
    caps = [cfg.cap_gpu_pages, max(0, mid_ids - slack), cfg.cap_cpu_pages]
    sim = W.SimTiers(cfg, seed, pool_ids, caps)
    r = TierRunner(cfg, seed, mid_ids, staging_bytes=max(sh.page_bytes * 3, 1 << 20))
    r.host.zero_()
    pool_m = np.zeros(sh.n_layers * pool_ids[0] * sh.chunk_bytes, np.uint8)
    mid_m = np.zeros(mid_ids * sh.page_bytes, np.uint8)
    host_m = np.zeros(pool_ids[2] * sh.page_bytes, np.uint8)
    pairs, moved, joins = set(), 0, 0
    for e in range(epochs):
        plan = sim.begin_epoch()
        want = oracle.rank_partition_tiers(plan.iota, plan.kv_pages, caps, plan.prev_tier)
        got = r.place(plan.iota, plan.kv_pages, plan.prev_tier, caps)
        for k in ("order", "tier", "bounds", "used"):
            assert np.array_equal(got[k], want[k]), (e, k)
        for k in range(2):
            assert np.array_equal(got["moves"][k], want["moves"][k]), (e, "moves", k)
        sim.apply_placement(got["tier"], got["moves"])
        r.execute(plan)
        oracle_apply_moves(plan.ops, sh, pool_m, mid_m, host_m)
        sim.end_epoch()
        r.fill(plan.fills)
        pv = pool_m.reshape(sh.n_layers, pool_ids[0], sh.chunk_bytes)
        for uid, first, pages in plan.fills:
            for j, g in enumerate(pages):
                pv[:, g] = W.page_content(seed, uid, first + j, sh)
        assert np.array_equal(r.pool.cpu().numpy(), pool_m), (e, "GPU pool")
        assert np.array_equal(r.mid.cpu().numpy(), mid_m), (e, "middle arena")
        assert np.array_equal(r.host.numpy(), host_m), (e, "host arena")
        joins += sum(1 for op in plan.ops if op[0] == "sync_all")
        for op in plan.ops:
            if op[0] == "move":
                pairs.add((op[2], op[3]))
                moved += len(op[4])
    r.close()
    assert moved > 0 and {(0, 1), (1, 0), (1, 2)} <= pairs, pairs
    if slack_div == 0:
        assert joins > 0
