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
