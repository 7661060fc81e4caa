"""numpy restatement of the oracle (TEST INFRASTRUCTURE -- see oracle/__init__.py).

A second, independent statement of the definitions in oracle.c, made of library routines
(``np.argsort(kind="stable")``, ``np.cumsum``, ``np.searchsorted``, fancy indexing) so that the
C oracle is pinned to something other than itself.  Citations as in oracle.c.
"""
import numpy as np


def sort_key(iota):
    """Canonical float key: -0 -> +0 (float ==, R12); NaN -> +inf bucket after +inf (R11)."""
    x = np.asarray(iota, dtype=np.float32).astype(np.float64)   # exact widening
    x = x + 0.0                                                 # -0.0 + 0.0 == +0.0
    nan = np.isnan(x)
    return np.where(nan, 0.0, x), nan


def rank(iota):
    """Programs in rank order: ascending idleness, ties by index, NaN last."""
    x, nan = sort_key(iota)
    # lexsort: last key is primary.  primary = is-NaN, then value; stable => ties by index.
    return np.lexsort((x, nan)).astype(np.int32)


def rank_partition(iota, s, prev_tier, cap_gpu, cap_cpu):
    s = np.asarray(s, dtype=np.int64)
    n = s.shape[0]
    if (s < 0).any() or cap_gpu < 0 or cap_cpu < 0:
        raise ValueError("negative size or capacity")
    order = rank(iota)
    incl = np.cumsum(s[order])                                  # inclusive prefix sums, int64
    # largest b with sum_{r<b} s <= C  ==  number of inclusive sums <= C (sums are non-decreasing)
    b_gpu = int(np.searchsorted(incl, cap_gpu, side="right"))
    base = int(incl[b_gpu - 1]) if b_gpu > 0 else 0
    b_cpu = int(np.searchsorted(incl, base + cap_cpu, side="right"))
    b_cpu = max(b_cpu, b_gpu)
    tier = np.full(n, 2, np.uint8)
    tier[order[:b_gpu]] = 0
    tier[order[b_gpu:b_cpu]] = 1
    used = np.array([base, (int(incl[b_cpu - 1]) if b_cpu > 0 else 0) - base], np.int64)
    out = dict(order=order, tier=tier, bounds=np.array([b_gpu, b_cpu], np.int32), used=used)
    if prev_tier is not None:
        prev = np.asarray(prev_tier, dtype=np.uint8)
        prev = np.where(prev > 2, 2, prev)
        was, now = prev[order], tier[order]
        asc, desc = order, order[::-1]
        wa, na, wd, nd = was, now, was[::-1], now[::-1]
        out["lists"] = [
            desc[(wd == 0) & (nd == 1)],      # demote, most idle first
            asc[(wa == 1) & (na == 0)],       # promote, least idle first
            desc[(wd != 2) & (nd == 2)],      # drop
            asc[(wa == 2) & (na == 0)],       # admit
            asc[(wa == 2) & (na == 1)],       # reserve
        ]
    return out


def demote(n_layers, chunk, pool, arena, gpu_pages, host_slots):
    """arena[h_j, l] = pool[l, g_j]  for all j, l  (fancy-index statement of oracle_demote)."""
    pv = pool.reshape(n_layers, -1, chunk)
    av = arena.reshape(-1, n_layers, chunk)
    g = np.asarray(gpu_pages, dtype=np.int64)
    h = np.asarray(host_slots, dtype=np.int64)
    av[h] = pv[:, g].transpose(1, 0, 2)


def promote(n_layers, chunk, pool, arena, host_slots, gpu_pages):
    pv = pool.reshape(n_layers, -1, chunk)
    av = arena.reshape(-1, n_layers, chunk)
    g = np.asarray(gpu_pages, dtype=np.int64)
    h = np.asarray(host_slots, dtype=np.int64)
    pv[:, g] = av[h].transpose(1, 0, 2)


# ------------------------------------------------------------------------------------------------
# NEXT-1: sticky, status-aware tier management restated with sorts and prefix sums
# ------------------------------------------------------------------------------------------------
ACTING, READY, NEW = 1, 2, 4


def move_slots(page_bytes, src, dst, src_slots, dst_slots):
    """Arena -> arena as one fancy-index assignment of whole page slots."""
    sv = src.reshape(-1, page_bytes)
    dv = dst.reshape(-1, page_bytes)
    dv[np.asarray(dst_slots, dtype=np.int64)] = sv[np.asarray(src_slots, dtype=np.int64)]


def sticky_rebalance(iota, s, prev_tier, flags, cap_gpu, cap_cpu):
    """Second statement of oracle_sticky_rebalance: instead of picking one victim / one candidate
    at a time it sorts each group once by the paper's priority and cuts the sorted list with a
    prefix sum (the cuts are monotone because sizes are non-negative)."""
    s = np.asarray(s, dtype=np.int64)
    prev = np.asarray(prev_tier, dtype=np.uint8)
    prev = np.where(prev > 2, 2, prev)
    flags = np.asarray(flags, dtype=np.uint8)
    n = s.shape[0]
    pos = np.empty(n, np.int64)
    pos[rank(iota)] = np.arange(n)                  # position in the total order (0 = least idle)
    tier = prev.copy()
    lazy = np.zeros(n, np.uint8)
    usage_gpu, usage_cpu = int(s[prev == 0].sum()), int(s[prev == 1].sum())
    if usage_cpu > cap_cpu or (s < 0).any() or cap_gpu < 0 or cap_cpu < 0:
        raise ValueError("bad argument")
    # demotion: victims in order (Acting first, then most idle first) until the rest fits
    g = np.flatnonzero(prev == 0)
    acting = (flags[g] & ACTING) != 0
    g = g[np.lexsort((-pos[g], ~acting))]           # primary: acting first; then descending position
    freed = np.cumsum(s[g])                         # pages freed after demoting the first k+1 victims
    # smallest v with usage - freed[v-1] <= cap  ==  number of k with usage - (freed before k) > cap
    before_k = freed - s[g]
    v = int(np.count_nonzero(usage_gpu - before_k > cap_gpu)) if usage_gpu > cap_gpu else 0
    victims = g[:v]
    demote, drop = [], []
    for p in victims:                               # CPU if it fits, else Waiting: per victim, in order
        if (flags[p] & ACTING) == 0:
            lazy[p] = 1
        usage_gpu -= int(s[p])
        if usage_cpu + int(s[p]) <= cap_cpu:
            tier[p] = 1; usage_cpu += int(s[p]); demote.append(p)
        else:
            tier[p] = 2; drop.append(p)
    # promotion: candidates sorted by (class, [size for class 3], position); longest prefix that fits
    ready = (flags & READY) != 0
    cls = np.where(prev == 1, 1, np.where((flags & NEW) != 0, 3, 2))
    c = np.flatnonzero(ready & (prev != 0))
    size_key = np.where(cls[c] == 3, s[c], 0)
    c = c[np.lexsort((pos[c], size_key, cls[c]))]
    k = int(np.searchsorted(np.cumsum(s[c]), cap_gpu - usage_gpu, side="right"))
    promote = [p for p in c[:k] if prev[p] == 1]
    admit = [p for p in c[:k] if prev[p] != 1]
    tier[c[:k]] = 0
    usage_gpu += int(s[c[:k]].sum())
    usage_cpu -= int(s[promote].sum()) if promote else 0
    i32 = lambda x: np.asarray(x, dtype=np.int32)
    return dict(tier=tier, lazy=lazy, used=np.array([usage_gpu, usage_cpu], np.int64),
                lists=[i32(demote), i32(promote), i32(drop), i32(admit), i32([])])


# ------------------------------------------------------------------------------------------------
# NEXT-3: typed eviction order as one lexsort
# ------------------------------------------------------------------------------------------------
def eviction_order(which_tier, page_owner, program_tier, last_access):
    """Resident pages, first to evict first: type priority (reversed between the tiers), then LRU,
    then page id."""
    owner = np.asarray(page_owner, dtype=np.int64)
    ptier = np.asarray(program_tier, dtype=np.int64)
    last = np.asarray(last_access, dtype=np.int64)
    pages = np.flatnonzero(owner >= 0)
    t = ptier[owner[pages]]
    # GPU HBM: inactive, idle, busy.  CPU DRAM: inactive, busy, idle.
    table = np.array([2, 1], np.int64) if which_tier == 0 else np.array([1, 2], np.int64)
    prio = np.where(t <= 1, table[np.minimum(t, 1)], 0)
    return pages[np.lexsort((pages, last[pages], prio))].astype(np.int32)


# ------------------------------------------------------------------------------------------------
# NEXT-4(i): Best-Fit-Decreasing of Waiting-queue promotions across replicas
# ------------------------------------------------------------------------------------------------
def bfd_assign(size, iota, flags, free_pages):
    """Largest candidate first (ties: returning before new, least idle, index); each goes to the
    replica with the most free pages if it fits there, else stays in Waiting (-1)."""
    size = np.asarray(size, dtype=np.int64)
    flags = np.asarray(flags, dtype=np.uint8)
    free = np.asarray(free_pages, dtype=np.int64).copy()
    m = size.shape[0]
    pos = np.empty(m, np.int64)
    pos[rank(iota)] = np.arange(m)
    order = np.lexsort((pos, (flags & NEW) != 0, -size))
    rep = np.full(m, -1, np.int32)
    for i in order:
        r = int(np.argmax(free))                      # first maximum = lowest replica index
        if size[i] <= free[r]:
            rep[i] = r
            free[r] -= size[i]
    return rep, free


# ------------------------------------------------------------------------------------------------
# NEXT-4(ii): the partition with T capacities
# ------------------------------------------------------------------------------------------------
def rank_partition_tiers(iota, s, caps, prev_tier=None):
    s = np.asarray(s, dtype=np.int64)
    n = s.shape[0]
    order = rank(iota)
    incl = np.cumsum(s[order])
    tier = np.full(n, len(caps), np.uint8)
    bounds, used, b, base = [], [], 0, 0
    for t, c in enumerate(caps):
        nb = max(b, int(np.searchsorted(incl, base + int(c), side="right")))
        tier[order[b:nb]] = t
        top = int(incl[nb - 1]) if nb > 0 else 0
        used.append(top - base if nb > b else 0)
        base = top if nb > b else base
        b = nb
        bounds.append(b)
    out = dict(order=order, tier=tier, bounds=np.array(bounds, np.int32), used=np.array(used, np.int64))
    if prev_tier is not None:
        was = np.minimum(np.asarray(prev_tier, dtype=np.int64), len(caps))
        now = tier.astype(np.int64)
        desc = order[::-1]
        out["moves"] = [desc[now[desc] > was[desc]].astype(np.int32),       # down: most idle first
                        order[now[order] < was[order]].astype(np.int32)]    # up: least idle first
    return out
