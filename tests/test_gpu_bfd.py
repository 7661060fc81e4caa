"""Parity of mori_bfd_assign (CUDA, through the C ABI) with the Best-Fit-Decreasing oracle
(P:L208-210): identical replica per candidate and identical free pages left."""
import numpy as np
import pytest
import torch

import oracle
from test_oracle_bfd_pins import rand_bfd_case, _gold

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(mori):
    pool = torch.zeros(2 * 4 * 8192, dtype=torch.uint8, device="cuda")
    m = mori.Mori(2, 2, 64, 16, pool)
    yield m
    m.close()


def gpu_bfd(m, size, iota, flags, free):
    d = "cuda"
    n = len(size)
    t = [torch.from_numpy(np.ascontiguousarray(x, dtype=dt)).to(d)
         for x, dt in ((size, np.int32), (iota, np.float32), (flags, np.uint8), (free, np.int64))]
    rep = torch.full((max(n, 1),), -9, dtype=torch.int32, device=d)
    left = torch.full((len(free),), -9, dtype=torch.int64, device=d)
    m.mori_bfd_assign(t[0], t[1], t[2], t[3], rep, left)
    torch.cuda.synchronize()
    return rep.cpu().numpy()[:n], left.cpu().numpy()


def test_hand_worked_packing(ctx):
    g = _gold()
    rep, left = gpu_bfd(ctx, g["size"], g["iota"], g["flags"], g["free"])
    assert rep.tolist() == g["replica"].astype(int).tolist() and left.tolist() == g["free_out"].astype(int).tolist()


@pytest.mark.parametrize("m,R", [(0, 1), (1, 1), (2, 32), (33, 3), (500, 8), (1024, 2), (1025, 5), (4096, 8),
                                 (8192, 32), (3000, 1)])
def test_random_queues_identical_packing(ctx, m, R):
    rng = np.random.default_rng(m * 37 + R)
    for rep_i in range(5):
        case = rand_bfd_case(rng, m, R)
        got, want = gpu_bfd(ctx, *case), oracle.bfd_assign(*case)
        assert np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1]), (m, R, rep_i)


def test_free_out_may_alias_free_pages_and_errors(ctx, mori):
    size = torch.tensor([4, 9, 2], dtype=torch.int32, device="cuda")
    iota = torch.tensor([0.1, 0.2, 0.3], dtype=torch.float32, device="cuda")
    flags = torch.tensor([2, 2, 6], dtype=torch.uint8, device="cuda")
    free = torch.tensor([5, 9], dtype=torch.int64, device="cuda")
    rep = torch.empty(3, dtype=torch.int32, device="cuda")
    ctx.mori_bfd_assign(size, iota, flags, free, rep, free)
    torch.cuda.synchronize()
    assert rep.tolist() == [0, 1, -1] and free.tolist() == [1, 0]
    with pytest.raises(mori.MoriError) as e:
        ctx.mori_bfd_assign(size, iota, flags, torch.zeros(33, dtype=torch.int64, device="cuda"), rep,
                            torch.zeros(33, dtype=torch.int64, device="cuda"))
    assert e.value.code == mori.ERR_UNSUPPORTED


def test_capacities_beyond_int32_take_the_wide_walk(ctx):
    rng = np.random.default_rng(3)
    size, iota, flags, _ = rand_bfd_case(rng, 500, 4)
    free = np.array([2 ** 40, 2 ** 33 + 5, 17, 2 ** 40], np.int64)
    got, want = gpu_bfd(ctx, size, iota, flags, free), oracle.bfd_assign(size, iota, flags, free)
    assert np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1])
