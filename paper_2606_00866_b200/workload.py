"""Seeded synthetic inputs for the MORI hot path: configs, agent trace, page contents, allocator.

This module is the ONE piece shared by the CPU oracle's tests and the CUDA path's tests/bench.
It holds no ranking, no partition and no page movement.  It makes inputs (idleness scores, KV
sizes, page tables, page bytes) and turns a placement that SOMEONE ELSE computed into page/slot
tables and call lists.  It imports neither ``oracle`` nor the CUDA binding.  One formula of the
paper does live here, because the trace must produce the hot path's input: ``windowed_idleness``,
Eq. (1) in float64.  Neither ``oracle/oracle.c`` nor ``csrc/idleness.cuh`` calls or shares it (each
states Eq. (1) itself); the oracle's pins use it as one more independent evaluation.

Recipe (BASELINE.json ``configs``): the paper replays private coding-agent
traces that are not available; a two-phase synthetic trace stands in, shaped by what
the paper states: persistent busy/idle phases, short tool calls of ~seconds and long
ones of ~a minute, tens of steps per program, closed-loop clients, a 5 s
scheduler tick and the windowed idleness of Eq. (1) with k = 5.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional, Tuple

import numpy as np

TIER_GPU, TIER_CPU, TIER_WAIT = 0, 1, 2
FLAG_ACTING, FLAG_READY, FLAG_NEW = 1, 2, 4     # inputs of the sticky policy mode
K_WINDOW = 5          # P:L194 "we use k=5 in all experiments"
TICK_S = 5.0          # P:L229 control-loop period


# --------------------------------------------------------------------------------------------
# configs
# --------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class KVShape:
    n_layers: int
    n_kv_heads: int
    head_dim: int
    page_tokens: int
    elem_bytes: int = 2      # bf16

    @property
    def chunk_bytes(self) -> int:
        """Contiguous bytes of one (layer, physical page): [K/V][kv_heads][page_tokens][head_dim]."""
        return 2 * self.n_kv_heads * self.page_tokens * self.head_dim * self.elem_bytes

    @property
    def page_bytes(self) -> int:
        return self.n_layers * self.chunk_bytes


@dataclass(frozen=True)
class Config:
    name: str
    index: int
    shape: KVShape
    n_programs: int
    gpu_pool_pages: int          # physical pages in the device pool
    cpu_pool_pages: int          # physical slots in the host arena
    epochs: int
    ctx_kind: str                # "uniform" | "lognormal"
    ctx_lo: int
    ctx_hi: int
    ctx_median: int = 0
    ctx_sigma: float = 0.8
    grow_lo: int = 0             # tokens added per completed step (cfg 2)
    grow_hi: int = 0
    f_busy: float = 0.5          # stationary busy fraction (cfg 3 sweeps it)
    iid_idleness: bool = False   # cfg 5: scores redrawn i.i.d. lognormal(0,1) every epoch
    random_pages: bool = False   # cfg 5: page tables randomly permuted across the pool
    scale: int = 1               # pools and contexts divided by this (SURVEY 8d scale rule)
    gpu_headroom_frac: float = 0.125   # physical pool kept free of the capacity the ranker sees

    @property
    def max_program_pages(self) -> int:
        return -(-self.ctx_hi // self.shape.page_tokens)

    @property
    def cap_gpu_pages(self) -> int:
        """Capacity handed to rank_partition: the physical pool minus headroom, so that
        promotions can start before the demotions that make room have finished."""
        return self.gpu_pool_pages - int(self.gpu_pool_pages * self.gpu_headroom_frac)

    @property
    def cap_cpu_pages(self) -> int:
        """Physical arena minus one largest program, so a demotion always finds free slots."""
        return max(0, self.cpu_pool_pages - self.max_program_pages)


_GIB = 1 << 30


def _pages(gib: int, shape: KVShape) -> int:
    return (gib * _GIB) // shape.page_bytes


def get_config(index: int, scale: int = 1, f_busy: Optional[float] = None) -> Config:
    """The five BASELINE.json configs (1-based).  ``scale`` divides both pools and all context
    lengths (keeping L/H/D/T/n) -- the scaled twins used where full-size mirrors do not fit."""
    if index == 1:
        sh = KVShape(2, 2, 64, 16)
        c = Config("cfg1-tiny", 1, sh, 8, 64, 256, 20, "uniform", 32, 400,
                   gpu_headroom_frac=0.0)
    elif index == 2:
        sh = KVShape(32, 8, 128, 16)
        c = Config("cfg2-llama3-8b", 2, sh, 64, _pages(60, sh), _pages(128, sh), 200,
                   "lognormal", 2048, 65536, 16384, 0.8, 500, 3000)
    elif index == 3:
        sh = KVShape(64, 8, 128, 16)
        c = Config("cfg3-qwen-32b", 3, sh, 128, _pages(80, sh), _pages(160, sh), 200,
                   "lognormal", 8192, 131072, 24576, 0.8)
    elif index == 4:
        sh = KVShape(80, 8, 128, 32)
        c = Config("cfg4-llama3-70b", 4, sh, 256, _pages(100, sh), _pages(200, sh), 100,
                   "lognormal", 4096, 131072, 32768, 0.8)
    elif index == 5:
        sh = KVShape(32, 8, 128, 16)
        c = Config("cfg5-frag", 5, sh, 4096, _pages(60, sh), _pages(128, sh), 500,
                   "uniform", 256, 8192, iid_idleness=True, random_pages=True)
    else:
        raise ValueError("config index must be 1..5")
    if f_busy is not None:
        c = replace(c, f_busy=f_busy, name=f"{c.name}-f{f_busy:g}")
    if scale != 1:
        T = c.shape.page_tokens
        c = replace(c, scale=scale, name=f"{c.name}/s{scale}",
                    gpu_pool_pages=c.gpu_pool_pages // scale,
                    cpu_pool_pages=c.cpu_pool_pages // scale,
                    ctx_lo=max(T, c.ctx_lo // scale), ctx_hi=max(T, c.ctx_hi // scale),
                    ctx_median=max(T, c.ctx_median // scale) if c.ctx_median else 0,
                    grow_lo=c.grow_lo // scale, grow_hi=max(c.grow_hi // scale, c.grow_lo // scale))
    return c


def config_seed(seed: int, cfg: Config) -> int:
    return seed * 10 + cfg.index


# --------------------------------------------------------------------------------------------
# Eq. (1): windowed idleness (input to the hot path; computed in float64, rounded once to f32)
# --------------------------------------------------------------------------------------------
def windowed_idleness(reasoning: np.ndarray, acting: np.ndarray) -> np.float32:
    """iota = T_act^(k) / (T_reason^(k) + T_act^(k)) over the given window (Eq. 1).

    ``reasoning`` / ``acting`` hold the durations of the last k cycles, the unfinished one
    included with its elapsed time; gated time was never added to either."""
    ta = float(np.sum(np.asarray(acting, dtype=np.float64)))
    tr = float(np.sum(np.asarray(reasoning, dtype=np.float64)))
    if ta + tr == 0.0:
        return np.float32(np.nan)
    return np.float32(ta / (tr + ta))


# --------------------------------------------------------------------------------------------
# trace generator
# --------------------------------------------------------------------------------------------
class Trace:
    """Closed-loop two-phase agent trace.  ``advance(tier)`` moves wall time by one tick and
    returns (idleness f32[n], context tokens i64[n], replaced bool[n])."""

    BUSY_MEDIAN_S, IDLE_MEDIAN_S, TOOL_SIGMA = 2.0, 60.0, 1.0      # BASELINE.json; sigma: DESIGN R13
    REASON_MEDIAN_S, REASON_SIGMA = 4.0, 0.5
    FLIP_RATE = 0.2

    def __init__(self, cfg: Config, seed: int):
        self.cfg = cfg
        self.rng = np.random.Generator(np.random.PCG64(config_seed(seed, cfg)))
        n = cfg.n_programs
        f = cfg.f_busy
        # mean flip rate stays 0.2 while the stationary busy fraction is f (cfg 3 sweep)
        self.p_busy_to_idle = 2 * self.FLIP_RATE * (1 - f)
        self.p_idle_to_busy = 2 * self.FLIP_RATE * f
        self.tokens = np.zeros(n, np.int64)
        self.uid = np.arange(n, dtype=np.int64)
        self._next_uid = n
        self.busy = np.zeros(n, bool)
        self.state = np.zeros(n, np.int8)           # 0 reasoning (or gated), 1 acting
        self.remaining = np.zeros(n, np.float64)    # time left in the current interval
        self.cur_reason = np.zeros(n, np.float64)   # elapsed in the unfinished cycle
        self.cur_act = np.zeros(n, np.float64)
        self.hist_reason = [[] for _ in range(n)]   # completed cycles, most recent last
        self.hist_act = [[] for _ in range(n)]
        self.steps_left = np.zeros(n, np.int64)
        # what a router would report to a device-side idleness tracker, in order:
        # (program, kind, reasoning s, acting s) with kind 0 = completed cycle, 1 = slot reset
        self.events: List[Tuple[int, int, float, float]] = []
        for p in range(n):
            self._spawn(p, new_uid=False)

    # -- draws -------------------------------------------------------------------------------
    def _draw_ctx(self) -> int:
        c = self.cfg
        if c.ctx_kind == "uniform":
            return int(self.rng.integers(c.ctx_lo, c.ctx_hi + 1))
        x = self.rng.lognormal(np.log(c.ctx_median), c.ctx_sigma)
        return int(min(max(int(x), c.ctx_lo), c.ctx_hi))

    def _draw_tool(self, p: int) -> float:
        med = self.BUSY_MEDIAN_S if self.busy[p] else self.IDLE_MEDIAN_S
        return float(self.rng.lognormal(np.log(med), self.TOOL_SIGMA))

    def _draw_reason(self) -> float:
        return float(self.rng.lognormal(np.log(self.REASON_MEDIAN_S), self.REASON_SIGMA))

    def _spawn(self, p: int, new_uid: bool = True):
        if new_uid:
            self.uid[p] = self._next_uid
            self._next_uid += 1
        self.tokens[p] = self._draw_ctx()
        self.busy[p] = self.rng.random() < self.cfg.f_busy
        # one synthetic completed cycle from the initial phase, so iota is never 0/0 (DESIGN R10)
        self.hist_reason[p] = [self._draw_reason()]
        self.hist_act[p] = [self._draw_tool(p)]
        self.events.append((p, 1, 0.0, 0.0))
        self.events.append((p, 0, self.hist_reason[p][0], self.hist_act[p][0]))
        self.cur_reason[p] = 0.0
        self.cur_act[p] = 0.0
        self.state[p] = 0
        self.remaining[p] = self._draw_reason()
        self.steps_left[p] = int(self.rng.integers(20, 61))

    # -- one tick ----------------------------------------------------------------------------
    def take_events(self):
        """-> (prog i32[m], kind u8[m], reasoning f64[m], acting f64[m]) since the last call, plus
        the open cycle's elapsed (reasoning f64[n], acting f64[n]) -- the inputs of Eq. (1)."""
        ev, self.events = self.events, []
        cols = list(zip(*ev)) if ev else [(), (), (), ()]
        return (np.array(cols[0], np.int32), np.array(cols[1], np.uint8), np.array(cols[2], np.float64),
                np.array(cols[3], np.float64), self.cur_reason.copy(), self.cur_act.copy())

    def advance(self, tier: np.ndarray) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
        cfg = self.cfg
        n = cfg.n_programs
        replaced = np.zeros(n, bool)
        if cfg.iid_idleness:
            iota = self.rng.lognormal(0.0, 1.0, n).astype(np.float32)
            return iota, self.tokens.copy(), replaced
        for p in range(n):
            dt = TICK_S
            while dt > 0.0:
                if self.state[p] == 0:                       # wants to reason
                    if tier[p] != TIER_GPU:
                        break                                # gated: time excluded
                    use = min(dt, self.remaining[p])
                    self.cur_reason[p] += use
                    self.remaining[p] -= use
                    dt -= use
                    if self.remaining[p] <= 0.0:             # inference step done
                        grow = int(self.rng.integers(cfg.grow_lo, cfg.grow_hi + 1)) if cfg.grow_hi else 0
                        self.steps_left[p] -= 1
                        if self.steps_left[p] <= 0 or self.tokens[p] + grow > cfg.ctx_hi:
                            self._spawn(p)                   # closed loop: a fresh program
                            replaced[p] = True
                            break
                        self.tokens[p] += grow
                        flip = self.p_busy_to_idle if self.busy[p] else self.p_idle_to_busy
                        if self.rng.random() < flip:
                            self.busy[p] = not self.busy[p]
                        self.state[p] = 1
                        self.remaining[p] = self._draw_tool(p)
                else:                                        # tool call runs whatever the tier
                    use = min(dt, self.remaining[p])
                    self.cur_act[p] += use
                    self.remaining[p] -= use
                    dt -= use
                    if self.remaining[p] <= 0.0:             # cycle closes
                        self.events.append((p, 0, float(self.cur_reason[p]), float(self.cur_act[p])))
                        self.hist_reason[p] = (self.hist_reason[p] + [self.cur_reason[p]])[-K_WINDOW:]
                        self.hist_act[p] = (self.hist_act[p] + [self.cur_act[p]])[-K_WINDOW:]
                        self.cur_reason[p] = 0.0
                        self.cur_act[p] = 0.0
                        self.state[p] = 0
                        self.remaining[p] = self._draw_reason()
        iota = np.empty(n, np.float32)
        for p in range(n):
            open_cycle = (self.cur_reason[p] + self.cur_act[p]) > 0.0
            k_done = K_WINDOW - 1 if open_cycle else K_WINDOW
            r = self.hist_reason[p][-k_done:] + ([self.cur_reason[p]] if open_cycle else [])
            a = self.hist_act[p][-k_done:] + ([self.cur_act[p]] if open_cycle else [])
            iota[p] = windowed_idleness(np.array(r), np.array(a))
        return iota, self.tokens.copy(), replaced


# --------------------------------------------------------------------------------------------
# page contents: counter-based generator G(seed, uid, logical page, layer, element)
# --------------------------------------------------------------------------------------------
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
    x = ((x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    x = ((x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
    return x ^ (x >> np.uint64(31))


def _f32_to_bf16_bits(f: np.ndarray) -> np.ndarray:
    u = f.astype(np.float32).view(np.uint32)
    return ((u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)).astype(np.uint32)


def page_key(seed: int, uid: int, logical_page: int) -> np.uint64:
    with np.errstate(over="ignore"):
        k = _splitmix64(np.array([np.uint64(seed & 0xFFFFFFFF) << np.uint64(32) ^ np.uint64(uid & 0xFFFFFFFF)],
                                 dtype=np.uint64))
        k = _splitmix64(k ^ np.uint64(logical_page))
    return k[0]


def page_keys(seed: int, uids: np.ndarray, logical_pages: np.ndarray) -> np.ndarray:
    """Vectorised page_key -> uint64[n] (what the device fill/check kernels take)."""
    with np.errstate(over="ignore"):
        u = (np.uint64(seed & 0xFFFFFFFF) << np.uint64(32)) ^ (np.asarray(uids).astype(np.uint64) & np.uint64(0xFFFFFFFF))
        return _splitmix64(_splitmix64(u) ^ np.asarray(logical_pages).astype(np.uint64))


def page_content(seed: int, uid: int, logical_page: int, shape: KVShape) -> np.ndarray:
    """uint8 [n_layers, chunk_bytes]: bf16 ~ N(0,1) (Irwin-Hall of 4 hash bytes), 2 values per
    64-bit hash.  Every byte is recomputable from (seed, uid, logical page, layer, offset)."""
    words = shape.chunk_bytes // 4                       # one uint32 = two bf16
    with np.errstate(over="ignore"):
        base = page_key(seed, uid, logical_page)
        ctr = (np.arange(shape.n_layers, dtype=np.uint64)[:, None] << np.uint64(32)) \
            + np.arange(words, dtype=np.uint64)[None, :]
        h = _splitmix64(base ^ ctr)
    out = np.zeros(h.shape, np.uint32)
    for half in range(2):
        s = np.zeros(h.shape, np.int32)
        for b in range(4):
            s += ((h >> np.uint64(8 * (4 * half + b))) & np.uint64(0xFF)).astype(np.int32)
        f = (s - 510).astype(np.float32) * np.float32(1.0 / 147.8)
        out |= _f32_to_bf16_bits(f) << np.uint32(16 * half)
    return out.view(np.uint8).reshape(shape.n_layers, shape.chunk_bytes)


# --------------------------------------------------------------------------------------------
# allocator + epoch planner
# --------------------------------------------------------------------------------------------
class IdAllocator:
    """Free-id set with a dependency tag per id (0 = free and clean; t > 0 = becomes free when
    move #t of the current epoch completes).  Lowest id first, or seeded-random (cfg 5)."""

    def __init__(self, n_ids: int, rng: Optional[np.random.Generator]):
        self.free = np.ones(n_ids, bool)
        self.tag = np.zeros(n_ids, np.int64)
        self.rng = rng

    def n_free(self, clean_only: bool = False) -> int:
        return int((self.free & (self.tag == 0)).sum()) if clean_only else int(self.free.sum())

    def alloc_run(self, k: int) -> Tuple[np.ndarray, int]:
        """k clean ids as ONE run of consecutive ids (first fit, lowest address) -- the
        "contiguous pinned host buffer" of a demoted program (BASELINE.json north_star; DESIGN
        R7).  Falls back to ``alloc(k, clean_only=True)`` (fragments) when no such run is free."""
        if k == 0:
            return np.zeros(0, np.int32), 0
        ok = self.free & (self.tag == 0)
        edges = np.diff(np.concatenate(([0], ok.view(np.int8), [0])))
        starts, ends = np.flatnonzero(edges == 1), np.flatnonzero(edges == -1)
        fit = np.flatnonzero(ends - starts >= k)
        if fit.size == 0:
            return self.alloc(k, clean_only=True)
        ids = np.arange(starts[fit[0]], starts[fit[0]] + k)
        self.free[ids] = False
        return ids.astype(np.int32), 0

    def alloc(self, k: int, clean_only: bool = False) -> Tuple[np.ndarray, int]:
        """-> (ids int32[k], max tag among them)."""
        if k == 0:
            return np.zeros(0, np.int32), 0
        cand = np.flatnonzero(self.free)
        clean = cand[self.tag[cand] == 0]
        if self.rng is not None:
            clean = self.rng.permutation(clean)
        if clean.size >= k:
            ids = clean[:k]
        else:
            if clean_only:
                raise MemoryError("not enough clean ids")
            dirty = cand[self.tag[cand] != 0]
            dirty = dirty[np.argsort(self.tag[dirty], kind="stable")]
            if clean.size + dirty.size < k:
                raise MemoryError("allocator exhausted")
            ids = np.concatenate([clean, dirty[:k - clean.size]])
        dep = int(self.tag[ids].max())
        self.last_tags = self.tag[ids].copy()       # per id: 0 = was clean, t = free once move #t completes
        self.free[ids] = False
        self.tag[ids] = 0
        return ids.astype(np.int32), dep

    def release(self, ids: np.ndarray, tag: int = 0):
        self.free[ids] = True
        self.tag[ids] = tag

    def clear_tags(self):
        self.tag[:] = 0


@dataclass
class EpochPlan:
    """What one epoch does, as tables.  ``ops`` is the issue order:
    ("demote", k, program, gpu_pages, host_slots)          k = 1, 2, ... within the epoch
    ("promote", 0, program, host_slots, gpu_pages, dep, first)   dep = k of the demote it must follow, or -1;
                                                           first = logical page of the program the lists start at
                                                           (a promotion is split by the demotion that frees its pages)
    ("sync_all",)                                          the host must join both streams here
    ``fills`` = [(uid, first_logical_page, gpu_pages)] executed after the epoch's sync."""
    iota: np.ndarray
    kv_pages: np.ndarray
    prev_tier: np.ndarray
    flags: Optional[np.ndarray] = None       # FLAG_* per program (sticky policy mode only)
    ops: list = field(default_factory=list)
    fills: list = field(default_factory=list)
    demote_pages: int = 0
    promote_pages: int = 0


def plan_calls(plan: "EpochPlan", merge: bool = True):
    """Turns the epoch's moves into the argument lists of the mover calls that will carry them.
    A move is a flat list of pages (include/mori.h), so the demotions of an epoch go out as ONE
    demote call per stretch of the plan that no promotion depends on, and the promotions likewise
    as one promote call per stretch with the same dependency: fewer calls, fewer ragged last staging
    segments, and the page order inside a call is the plan's (the paper's move order, P:L206 /
    L208).  ``merge=False``: one call per program.

    -> (steps, need_tickets); steps, in issue order:
         ("d", gpu_pages i32[], host_slots i32[], n, [k ...])   k = the plan's demote numbers it carries
         ("p", host_slots i32[], gpu_pages i32[], n, dep)       dep = demote number it must follow, or 0
         ("sync",)                                              the host joins both directions here
    A promotion's ``dep`` is always carried by a demote step issued BEFORE it."""
    steps = []
    dem, pro, pro_dep = [], [], 0
    flushed = set()

    def cat(parts):
        return np.ascontiguousarray(parts[0] if len(parts) == 1 else np.concatenate(parts), dtype=np.int32)

    def flush_dem():
        if dem:
            g, h = cat([o[3] for o in dem]), cat([o[4] for o in dem])
            steps.append(("d", g, h, g.size, [o[1] for o in dem]))
            flushed.update(o[1] for o in dem)
            dem.clear()

    def flush_pro():
        nonlocal pro_dep
        if pro:
            h, g = cat([o[3] for o in pro]), cat([o[4] for o in pro])
            steps.append(("p", h, g, g.size, pro_dep))
            pro.clear()
        pro_dep = 0

    for op in plan.ops:
        if op[0] == "demote":
            dem.append(op)
            if not merge:
                flush_dem()
        elif op[0] == "promote":
            dep = op[5] if op[5] > 0 else 0
            if pro and dep != pro_dep:        # a different dependency: its own call
                flush_pro()
            if dep > 0 and dep not in flushed:
                flush_dem()                   # the demotion it follows ends its call here, so the
                                              # promotion waits for that much and no more
            pro.append(op)
            pro_dep = dep
            if not merge:
                flush_pro()
        elif op[0] == "sync_all":
            flush_dem(); flush_pro()
            steps.append(("sync",))
            flushed.clear()
    # both directions start together: the demote call first (it is what vacates pages)
    flush_dem(); flush_pro()
    return steps, any(st[0] == "p" and st[4] > 0 for st in steps)


class Sim:
    """Epoch state machine: owns the trace, the per-program page/slot tables and the allocators.
    The placement itself comes from the caller (oracle or CUDA path)."""

    def __init__(self, cfg: Config, seed: int):
        self.cfg, self.seed = cfg, seed
        self.trace = Trace(cfg, seed)
        n = cfg.n_programs
        arng = np.random.Generator(np.random.PCG64(config_seed(seed, cfg) + 7919)) if cfg.random_pages else None
        self.gpu_alloc = IdAllocator(cfg.gpu_pool_pages, arng)     # cfg 5: every device page scattered
        self.cpu_alloc = IdAllocator(cfg.cpu_pool_pages, None)     # host buffers: contiguous runs first
        self.tier = np.full(n, TIER_WAIT, np.uint8)
        self.gpu_pages: List[np.ndarray] = [np.zeros(0, np.int32) for _ in range(n)]
        self.host_slots: List[np.ndarray] = [np.zeros(0, np.int32) for _ in range(n)]
        self.ever_resident = np.zeros(n, bool)      # has held KV on this replica (else "new arrival")
        self.epoch = 0
        self._pending = None

    def flags(self) -> np.ndarray:
        """Status inputs of the sticky policy: ACTING while a tool call runs,
        READY when the program wants inference (for a CPU/Waiting program: its request is gated
        and waiting), NEW until it has held KV once."""
        st = self.trace.state
        f = np.where(st == 1, FLAG_ACTING, FLAG_READY).astype(np.uint8)
        f[~self.ever_resident] |= FLAG_NEW
        return f

    # step 1: inputs of this epoch's placement
    def begin_epoch(self) -> EpochPlan:
        iota, tokens, replaced = self.trace.advance(self.tier)
        for p in np.flatnonzero(replaced):                   # finished program: KV gone, slot reused
            self._drop(p)
            self.tier[p] = TIER_WAIT
            self.ever_resident[p] = False
        T = self.cfg.shape.page_tokens
        kv_pages = ((tokens + T - 1) // T).astype(np.int32)
        plan = EpochPlan(iota=iota, kv_pages=kv_pages, prev_tier=self.tier.copy(), flags=self.flags())
        self._pending = plan
        return plan

    def _drop(self, p: int):
        if self.gpu_pages[p].size:
            self.gpu_alloc.release(self.gpu_pages[p])
            self.gpu_pages[p] = np.zeros(0, np.int32)
        if self.host_slots[p].size:
            self.cpu_alloc.release(self.host_slots[p])
            self.host_slots[p] = np.zeros(0, np.int32)

    # step 2: turn the placement (tier + lists, computed elsewhere) into tables
    def apply_placement(self, tier: np.ndarray, lists: List[np.ndarray]) -> EpochPlan:
        plan = self._pending
        demote, promote, drop = lists[0], lists[1], lists[2]
        for p in drop:                                       # P:L178 "discarded entirely"
            self._drop(int(p))
        dem_q = [int(p) for p in demote if self.gpu_pages[int(p)].size]   # else: labelled only
        pro_q = [int(p) for p in promote if self.host_slots[int(p)].size]  # else: "reserve" label (R9)
        ops, k = [], 0
        while dem_q or pro_q:
            progress = False
            while True:                                      # alternate, so both directions start at once
                did = False
                if dem_q and self.cpu_alloc.n_free(clean_only=True) >= self.gpu_pages[dem_q[0]].size:
                    p = dem_q.pop(0)
                    pages = self.gpu_pages[p]
                    slots, _ = self.cpu_alloc.alloc_run(pages.size)
                    k += 1
                    ops.append(("demote", k, p, pages.copy(), slots))
                    self.gpu_alloc.release(pages, tag=k)     # reusable once demote #k completes
                    self.host_slots[p] = slots
                    self.gpu_pages[p] = np.zeros(0, np.int32)
                    plan.demote_pages += int(pages.size)
                    did = True
                if pro_q and self.gpu_alloc.n_free() >= self.host_slots[pro_q[0]].size:
                    p = pro_q.pop(0)
                    slots = self.host_slots[p]
                    pages, dep = self.gpu_alloc.alloc(slots.size)
                    if dep > 0:
                        # some of the pages are still being vacated: the part that lands in clean
                        # pages goes at once, the rest follows the demotion that frees it, one piece
                        # per demotion, in the order the demotions complete
                        tags = self.gpu_alloc.last_tags              # non-decreasing along the logical pages
                        for t in np.unique(tags):
                            sel = np.flatnonzero(tags == t)
                            assert sel[-1] - sel[0] + 1 == sel.size     # a contiguous range of logical pages
                            ops.append(("promote", 0, p, slots[sel].copy(), pages[sel], int(t) if t > 0 else -1,
                                        int(sel[0])))
                    else:
                        ops.append(("promote", 0, p, slots.copy(), pages, -1, 0))
                    self.cpu_alloc.release(slots, tag=1)     # not reusable before the next join
                    self.gpu_pages[p] = pages
                    self.host_slots[p] = np.zeros(0, np.int32)
                    plan.promote_pages += int(slots.size)
                    did = True
                if not did:
                    break
                progress = True
            if dem_q or pro_q:
                if not progress:
                    raise MemoryError("placement does not fit the physical pools")
                ops.append(("sync_all",))                    # join both streams; frees become clean
                self.gpu_alloc.clear_tags()
                self.cpu_alloc.clear_tags()
        plan.ops = ops
        self.tier = np.asarray(tier, dtype=np.uint8).copy()
        return plan

    # step 3: after the movers have been joined
    def end_epoch(self) -> EpochPlan:
        plan = self._pending
        self.gpu_alloc.clear_tags()
        self.cpu_alloc.clear_tags()
        self.ever_resident |= self.tier == TIER_GPU
        for p in np.flatnonzero(self.tier == TIER_GPU):      # admit + growth: recompute prefill
            need = int(plan.kv_pages[p]) - self.gpu_pages[p].size
            if need > 0:
                new, _ = self.gpu_alloc.alloc(need)
                plan.fills.append((int(self.trace.uid[p]), int(self.gpu_pages[p].size), new))
                self.gpu_pages[p] = np.concatenate([self.gpu_pages[p], new])
        self.epoch += 1
        self._pending = None
        return plan


# --------------------------------------------------------------------------------------------
# more tiers (SURVEY 8f NEXT-4 ii): the same epoch state machine over a hierarchy
# --------------------------------------------------------------------------------------------
class SimTiers:
    """Epoch state machine for T storage tiers: tier 0 is the paged GPU pool, tiers 1 .. T-1 are
    page-major arenas from fast to slow (e.g. peer-GPU HBM, then host DRAM: the "intermediate tier"
    of P:L347), tier value T is Waiting.  Like ``Sim`` it holds none of the method's arithmetic:
    the placement (tier per program + the DOWN / UP move lists of a T-capacity partition) comes
    from the caller, and is turned into page / slot tables here.

    ``pool_ids[t]`` = physical pages / slots of tier t; ``caps[t]`` = the capacity the ranker is
    given (physical minus headroom, R23).  Ids freed by a move of this epoch are not
    handed out again before the next join ("sync_all"), so moves of one phase never alias and the
    movers need no cross-tier tickets."""

    def __init__(self, cfg: Config, seed: int, pool_ids: List[int], caps: List[int]):
        assert len(pool_ids) == len(caps) >= 1
        self.cfg, self.seed, self.T = cfg, seed, len(caps)
        self.pool_ids, self.caps = list(pool_ids), list(caps)
        self.trace = Trace(cfg, seed)
        n = cfg.n_programs
        arng = np.random.Generator(np.random.PCG64(config_seed(seed, cfg) + 7919)) if cfg.random_pages else None
        self.alloc = [IdAllocator(pool_ids[0], arng)] + [IdAllocator(k, None) for k in pool_ids[1:]]
        self.tier = np.full(n, self.T, np.uint8)
        self.where = np.full(n, -1, np.int64)               # tier that holds the program's bytes, -1: none
        self.ids: List[np.ndarray] = [np.zeros(0, np.int32) for _ in range(n)]
        self.epoch = 0
        self._pending = None

    def begin_epoch(self) -> EpochPlan:
        # the trace gates on "not in the GPU tier": tier 0 here as well
        iota, tokens, replaced = self.trace.advance(np.where(self.tier == 0, TIER_GPU, TIER_WAIT).astype(np.uint8))
        for p in np.flatnonzero(replaced):
            self._drop(int(p))
            self.tier[p] = self.T
        Tk = self.cfg.shape.page_tokens
        kv_pages = ((tokens + Tk - 1) // Tk).astype(np.int32)
        plan = EpochPlan(iota=iota, kv_pages=kv_pages, prev_tier=self.tier.copy())
        self._pending = plan
        return plan

    def _drop(self, p: int):
        if self.where[p] >= 0 and self.ids[p].size:
            self.alloc[self.where[p]].release(self.ids[p])
        self.ids[p] = np.zeros(0, np.int32)
        self.where[p] = -1

    def apply_placement(self, tier: np.ndarray, moves: List[np.ndarray]) -> EpochPlan:
        """``moves`` = [down (most idle first), up (least idle first)] as the T-capacity partition
        lists them.  plan.ops entries: ("move", program, from_tier, to_tier, src_ids, dst_ids) and
        ("sync_all",)."""
        plan = self._pending
        tier = np.asarray(tier, dtype=np.uint8)
        queue = []
        for p in list(moves[0]) + list(moves[1]):
            p = int(p)
            to = int(tier[p])
            if to >= self.T:                                 # P:L178 "discarded entirely"
                self._drop(p)
            elif self.where[p] >= 0 and self.where[p] != to and self.ids[p].size:
                queue.append((p, int(self.where[p]), to))
            # else: a label without bytes (R9); a GPU-tier one is filled in end_epoch
        ops, progressed_since_sync = [], True
        while queue:
            rest, did = [], False
            for p, frm, to in queue:
                k = int(self.ids[p].size)
                al = self.alloc[to]
                if al.n_free(clean_only=True) >= k:
                    dst, _ = al.alloc(k, clean_only=True) if to == 0 else al.alloc_run(k)
                    src = self.ids[p]
                    ops.append(("move", p, frm, to, src.copy(), dst))
                    self.alloc[frm].release(src, tag=1)      # not reusable before the next join
                    self.ids[p], self.where[p] = dst, to
                    plan.demote_pages += k if to > frm else 0
                    plan.promote_pages += k if to < frm else 0
                    did = True
                else:
                    rest.append((p, frm, to))
            queue = rest
            if did:
                progressed_since_sync = True
            elif queue:
                if not progressed_since_sync:
                    raise MemoryError("placement does not fit the physical pools")
                ops.append(("sync_all",))
                for al in self.alloc:
                    al.clear_tags()
                progressed_since_sync = False
        plan.ops = ops
        self.tier = tier.copy()
        return plan

    def end_epoch(self) -> EpochPlan:
        plan = self._pending
        for al in self.alloc:
            al.clear_tags()
        for p in np.flatnonzero(self.tier == 0):             # admit + growth: recompute prefill
            have = int(self.ids[p].size) if self.where[p] == 0 else 0
            need = int(plan.kv_pages[p]) - have
            if need > 0:
                new, _ = self.alloc[0].alloc(need)
                plan.fills.append((int(self.trace.uid[p]), have, new))
                self.ids[p] = np.concatenate([self.ids[p], new]) if have else new
                self.where[p] = 0
        self.epoch += 1
        self._pending = None
        return plan

    def resident(self):
        """-> per tier, [(uid, 0, ids)] of every program whose bytes live there."""
        out = [[] for _ in range(self.T)]
        for p in range(self.cfg.n_programs):
            if self.where[p] >= 0 and self.ids[p].size:
                out[self.where[p]].append((int(self.trace.uid[p]), 0, self.ids[p]))
        return out
