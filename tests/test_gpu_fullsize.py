"""Parity at BASELINE.json's full sizes, in the launch configurations bench.py times (cfg 2:
60 GiB device pool, 128 GiB pinned arena, AUTO paths, default staging; likewise cfg 3 and cfg 5, and
cfg 4 at the scale this box's host RAM allows): placement bit-exact
against the oracle every epoch; moved bytes checked on SAMPLED pages the oracle computes one by
one (first, last and random logical pages of every moved program), plus a property that holds at
any size: every resident page of both tiers still equals the counter-based generator."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_00866_b200 import workload as W
from paper_2606_00866_b200.harness import GpuRunner

pytestmark = pytest.mark.gpu
GIB = 1 << 30


def _mem_available():
    for line in open("/proc/meminfo"):
        if line.startswith("MemAvailable:"):
            return int(line.split()[1]) * 1024
    return 0


def _mem_total():
    for line in open("/proc/meminfo"):
        if line.startswith("MemTotal:"):
            return int(line.split()[1]) * 1024
    return 0


def _sample(n, rng, k=4):
    js = {0, n - 1} | {int(x) for x in rng.integers(0, n, size=min(k, n))}
    return sorted(js)


def _oracle_pages(seed, uid, js, sh, promote):
    """Expected bytes of logical pages ``js`` after a move, computed by the oracle's mover on a
    miniature pool/arena that holds exactly those pages (page j of the sample sits in mini pool
    page j' and mini slot j')."""
    k = len(js)
    pool = np.zeros(sh.n_layers * k * sh.chunk_bytes, np.uint8)
    arena = np.zeros(k * sh.page_bytes, np.uint8)
    ids = np.arange(k, dtype=np.int32)
    content = [W.page_content(seed, uid, j, sh) for j in js]          # [L, chunk] each
    if promote:
        arena.reshape(k, sh.n_layers, sh.chunk_bytes)[:] = np.stack(content)
        oracle.promote(sh.n_layers, sh.chunk_bytes, pool, arena, ids, ids[::-1].copy())
        pv = pool.reshape(sh.n_layers, k, sh.chunk_bytes)
        return [pv[:, k - 1 - i] for i in range(k)]                    # [L, chunk] per sampled page
    pool.reshape(sh.n_layers, k, sh.chunk_bytes)[:] = np.stack(content, axis=1)
    oracle.demote(sh.n_layers, sh.chunk_bytes, pool, arena, ids, ids[::-1].copy())
    av = arena.reshape(k, sh.n_layers, sh.chunk_bytes)
    return [av[k - 1 - i] for i in range(k)]


def _scale_that_fits(idx):
    """The smallest power-of-two scale whose pinned arena leaves 20 GiB of this box's RAM free."""
    scale = 1
    while True:
        cfg = W.get_config(idx, scale)
        if cfg.cpu_pool_pages * cfg.shape.page_bytes + 20 * GIB <= _mem_available():
            return scale
        scale *= 2


EPOCHS = 40


@pytest.mark.parametrize("idx,f_busy", [(2, None), (5, None), (3, 0.5), (4, None)])
def test_full_size_epochs_sampled_parity(mori, idx, f_busy):
    """The configurations bench.py launches: cfg 2, 3 and 5 as written (128 / 160 / 128 GiB pinned
    arenas fit a 196 GiB host), cfg 4 with pools and contexts halved (its 200 GiB arena does not)."""
    torch.cuda.empty_cache()
    scale = _scale_that_fits(idx)
    print(f"cfg {idx}: scale {scale} (MemAvailable {_mem_available() / GIB:.0f} GiB)")
    if idx in (2, 3, 5) and scale != 1:
        print(f"NOTE cfg {idx} does not run as written here: MemAvailable {_mem_available() / GIB:.0f} of "
              f"{_mem_total() / GIB:.0f} GiB leaves no room for its pinned arena; scale {scale}")
    seed = 866
    arena = None
    while arena is None:                               # a refused page-lock falls back to the next scale, and says so
        assert scale <= 8, "this box cannot pin even an eighth of the arena"
        cfg = W.get_config(idx, scale, f_busy)
        sh = cfg.shape
        arena_bytes = cfg.cpu_pool_pages * sh.page_bytes
        try:
            arena = mori.Mori.mori_host_alloc(arena_bytes)
        except mori.MoriError as e:
            print(f"NOTE cfg {idx} at scale {scale}: pinning {arena_bytes / GIB:.0f} GiB refused ({e}); trying scale {scale * 2}")
            scale *= 2
    assert arena.is_pinned()
    r = GpuRunner(cfg, seed, arena=arena)                  # AUTO paths, default staging = bench.py
    sim = W.Sim(cfg, seed)
    rng = np.random.default_rng(5)
    av = arena.numpy().reshape(cfg.cpu_pool_pages, sh.n_layers, sh.chunk_bytes)
    pv = r.pool.view(sh.n_layers, cfg.gpu_pool_pages, sh.chunk_bytes)
    moved = checked = 0
    for e in range(EPOCHS):
        plan = sim.begin_epoch()
        want = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        got = r.place(plan.iota, plan.kv_pages, plan.prev_tier)
        for k in ("order", "tier", "bounds", "used"):
            assert np.array_equal(got[k], want[k]), (e, k)
        for k in range(5):
            assert np.array_equal(got["lists"][k], want["lists"][k]), (e, "list", k)
        sim.apply_placement(got["tier"], got["lists"])
        r.execute(plan)
        for op in plan.ops:
            if op[0] not in ("demote", "promote"):
                continue
            uid = int(sim.trace.uid[op[2]])
            promote = op[0] == "promote"
            slots, pages = (op[3], op[4]) if promote else (op[4], op[3])
            first = op[6] if promote else 0                  # a promotion may cover a range of the program's pages
            js = _sample(len(pages), rng)
            exp = _oracle_pages(seed, uid, [first + j for j in js], sh, promote)
            for want_page, j in zip(exp, js):
                if promote:     # read the destination page back by a plain strided copy
                    have = pv[:, int(pages[j])].cpu().numpy()
                else:
                    have = av[int(slots[j])]
                assert np.array_equal(have, want_page), (e, op[0], op[2], j)
                checked += 1
            moved += len(pages)
        sim.end_epoch()
        r.fill(plan.fills)
    assert moved * sh.page_bytes > 8 * GIB // scale and checked > 40    # many GiB really moved
    gtri, htri = r.resident(sim)
    assert r.check(gtri) == 0, "a resident device page differs from the generator"
    assert r.check(htri, arena=True) == 0, "a resident host slot differs from the generator"
    r.close()
    mori.Mori.mori_host_free(arena)
