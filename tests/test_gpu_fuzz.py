"""Randomised call sequences through the C ABI against the oracle's memcpy movers: random KV
geometries, staging sizes and paths; demotions and promotions issued back to back with NO join
unless the sequence says so, every cross-direction hazard covered by the ticket the header asks
for (include/mori.h: calls of one direction take effect in issue order, the two directions are
ordered only by tickets).  After the final join both pools must equal the oracle's byte for byte."""
import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu


def _scenario(mori, seed):
    rng = np.random.default_rng(1000 + seed)
    L = int(rng.integers(1, 7))
    H = int(rng.integers(1, 9))
    D = int(rng.choice([8, 16, 32, 64, 128]))
    T = int(rng.integers(1, 33))
    chunk = 2 * H * T * D * 2                                   # always a multiple of 16
    page = L * chunk
    budget = 96 << 20                                            # bytes per pool, keeps a scenario fast
    P = int(np.clip(budget // page, 24, 700))
    S = int(np.clip(budget // page, 24, 700))
    path = int(rng.choice([0, 0, 0, 1, 2, 3]))                   # mostly AUTO (per-call choice)
    kernel = int(rng.choice([0, 1, 2]))
    staging = int(rng.choice([0, 3 * page, 17 * page, 64 * page]))
    g = torch.Generator(device="cpu").manual_seed(seed)
    pool_h = torch.randint(0, 256, (L * P * chunk,), dtype=torch.uint8, generator=g)
    arena = torch.randint(0, 256, (S * L * chunk,), dtype=torch.uint8, generator=g).pin_memory()
    pool = pool_h.cuda()
    m = mori.Mori(L, H, D, T, pool, arena, path_demote=path, path_promote=path, copy_kernel=kernel,
                  staging_bytes=staging)
    pool_m, arena_m = pool_h.numpy().copy(), arena.numpy().copy()
    # un-joined work: id -> ticket of the last call of that kind that touches it
    dem_reads_page, dem_writes_slot = {}, {}
    pro_reads_slot, pro_writes_page = {}, {}
    n_ops = int(rng.integers(6, 16))
    for _ in range(n_ops):
        kind = rng.choice(["demote", "promote", "sync"], p=[0.45, 0.45, 0.10])
        if kind == "sync":
            m.mori_sync(mori.BOTH)
            for d in (dem_reads_page, dem_writes_slot, pro_reads_slot, pro_writes_page):
                d.clear()
            continue
        k = int(rng.integers(0, min(P, S) // 2))
        if rng.random() < 0.3:
            k = int(rng.integers(0, 6))                          # small calls: the one-launch path under AUTO
        pages = rng.permutation(P)[:k].astype(np.int32)          # destination ids must be distinct
        if rng.random() < 0.5 and k:
            start = int(rng.integers(0, S - k + 1))
            slots = (start + np.arange(k)).astype(np.int32)      # one run of consecutive slots
        else:
            slots = rng.permutation(S)[:k].astype(np.int32)
        if kind == "demote":
            # reads pages (hazard: an un-joined promotion writes them), writes slots (hazard: an
            # un-joined promotion reads them): one ticket, everything of the call waits for it
            wait = max([pro_writes_page.get(int(x), 0) for x in pages] +
                       [pro_reads_slot.get(int(x), 0) for x in slots] + [0])
            t = m.mori_demote(pages, slots, wait_promote_ticket=wait)
            oracle.demote(L, chunk, pool_m, arena_m, pages, slots)
            for x in pages:
                dem_reads_page[int(x)] = t
            for x in slots:
                dem_writes_slot[int(x)] = t
        else:
            # writes pages (hazard: an un-joined demotion reads them -> pages_after_demote), reads
            # slots (hazard: an un-joined demotion writes them -> slots_after_demote)
            wp = max([dem_reads_page.get(int(x), 0) for x in pages] + [0])
            ws = max([dem_writes_slot.get(int(x), 0) for x in slots] + [0])
            t = m.mori_promote(slots, pages, pages_after_demote=wp, slots_after_demote=ws)
            oracle.promote(L, chunk, pool_m, arena_m, slots, pages)
            for x in pages:
                pro_writes_page[int(x)] = t
            for x in slots:
                pro_reads_slot[int(x)] = t
    m.mori_sync(mori.BOTH)
    ok_arena = np.array_equal(arena.numpy(), arena_m)
    ok_pool = np.array_equal(pool.cpu().numpy(), pool_m)
    m.close()
    return ok_arena, ok_pool, dict(L=L, H=H, D=D, T=T, P=P, S=S, path=path, kernel=kernel, staging=staging // page,
                                   n_ops=n_ops)


@pytest.mark.parametrize("block", range(6))
def test_random_call_sequences_match_the_oracle(mori, block):
    for seed in range(block * 8, block * 8 + 8):
        ok_arena, ok_pool, what = _scenario(mori, seed)
        assert ok_arena, ("arena differs", seed, what)
        assert ok_pool, ("pool differs", seed, what)
