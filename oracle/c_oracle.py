"""ctypes loader for oracle.c (TEST INFRASTRUCTURE -- see oracle/__init__.py)."""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def lib_path():
    return _LIB


def build(force=False):
    """Compile oracle.c with gcc (plain C11, no CUDA)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", "-std=c11", "-O2", "-Wall", "-Wextra", "-shared", "-fPIC",
                           _SRC, "-o", tmp])
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.oracle_rank_partition.argtypes = [i32, vp, vp, vp, i64, i64, vp, vp, vp, vp, vp, vp]
        L.oracle_rank_partition.restype = C.c_int
        L.oracle_bruteforce_partition.argtypes = [i32, vp, vp, i64, i64, vp, vp, vp]
        L.oracle_bruteforce_partition.restype = C.c_int
        L.oracle_sticky_rebalance.argtypes = [i32, vp, vp, vp, vp, i64, i64, vp, vp, vp, vp, vp]
        L.oracle_sticky_rebalance.restype = C.c_int
        L.oracle_rank_partition_tiers.argtypes = [i32, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp]
        L.oracle_rank_partition_tiers.restype = C.c_int
        L.oracle_bfd_assign.argtypes = [i32, vp, vp, vp, i32, vp, vp, vp]
        L.oracle_bfd_assign.restype = C.c_int
        L.oracle_eviction_order.argtypes = [i32, i64, vp, i32, vp, vp, vp, C.POINTER(i64)]
        L.oracle_eviction_order.restype = C.c_int
        L.oracle_idleness_update.argtypes = [i32, vp, vp, vp, i32, i64, vp, vp, vp, vp]
        L.oracle_idleness_update.restype = C.c_int
        L.oracle_idleness_eval.argtypes = [i32, vp, vp, vp, i32, vp, vp, vp]
        L.oracle_idleness_eval.restype = C.c_int
        L.oracle_move_slots.argtypes = [i64, vp, i64, vp, i64, i64, vp, vp]
        L.oracle_move_slots.restype = C.c_int
        for f in (L.oracle_demote, L.oracle_promote):
            f.argtypes = [i32, i64, vp, i64, vp, i64, i64, vp, vp]
            f.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def rank_partition(iota, s, prev_tier, cap_gpu, cap_cpu):
    """oracle_rank_partition -> dict(order, tier, bounds, used, lists (list of 5 arrays))."""
    iota = np.ascontiguousarray(iota, dtype=np.float32)
    s = np.ascontiguousarray(s, dtype=np.int32)
    n = int(iota.shape[0])
    assert s.shape == (n,)
    prev = None if prev_tier is None else np.ascontiguousarray(prev_tier, dtype=np.uint8)
    order = np.empty(n, np.int32)
    tier = np.empty(n, np.uint8)
    bounds = np.zeros(2, np.int32)
    used = np.zeros(2, np.int64)
    lists = np.full((5, max(n, 1)), -1, np.int32)[:, :n].copy() if n else np.zeros((5, 0), np.int32)
    counts = np.zeros(5, np.int32)
    rc = _load().oracle_rank_partition(n, _p(iota), _p(s), _p(prev), int(cap_gpu), int(cap_cpu),
                                       _p(order), _p(tier), _p(bounds), _p(used),
                                       _p(lists) if prev is not None else None,
                                       _p(counts) if prev is not None else None)
    if rc != 0:
        raise ValueError(f"oracle_rank_partition: bad argument (rc={rc})")
    out = dict(order=order, tier=tier, bounds=bounds, used=used)
    if prev is not None:
        out["lists"] = [lists[k, :counts[k]].copy() for k in range(5)]
    return out


def sticky_rebalance(iota, s, prev_tier, flags, cap_gpu, cap_cpu):
    """oracle_sticky_rebalance -> dict(tier, lazy, used, lists (5 arrays; reserve always empty))."""
    iota = np.ascontiguousarray(iota, dtype=np.float32)
    s = np.ascontiguousarray(s, dtype=np.int32)
    prev = np.ascontiguousarray(prev_tier, dtype=np.uint8)
    flags = np.ascontiguousarray(flags, dtype=np.uint8)
    n = int(iota.shape[0])
    assert s.shape == (n,) and prev.shape == (n,) and flags.shape == (n,)
    tier = np.empty(max(n, 1), np.uint8)
    lazy = np.zeros(max(n, 1), np.uint8)
    used = np.zeros(2, np.int64)
    lists = np.full((5, max(n, 1)), -1, np.int32)
    if n:
        lists = np.ascontiguousarray(lists[:, :n])
    counts = np.zeros(5, np.int32)
    rc = _load().oracle_sticky_rebalance(n, _p(iota), _p(s), _p(prev), _p(flags), int(cap_gpu),
                                         int(cap_cpu), _p(tier), _p(lazy), _p(used), _p(lists), _p(counts))
    if rc != 0:
        raise ValueError(f"oracle_sticky_rebalance: bad argument (rc={rc})")
    return dict(tier=tier[:n], lazy=lazy[:n], used=used,
                lists=[lists[k, :counts[k]].copy() for k in range(5)])


def rank_partition_tiers(iota, s, caps, prev_tier=None):
    """oracle_rank_partition_tiers -> dict(order, tier (T = waiting), bounds[T], used[T]) and, with
    ``prev_tier``, moves = [down (most idle first), up (least idle first)]."""
    iota = np.ascontiguousarray(iota, dtype=np.float32)
    s = np.ascontiguousarray(s, dtype=np.int32)
    caps = np.ascontiguousarray(caps, dtype=np.int64)
    prev = None if prev_tier is None else np.ascontiguousarray(prev_tier, dtype=np.uint8)
    n, T = iota.size, caps.size
    order = np.empty(max(n, 1), np.int32); tier = np.empty(max(n, 1), np.uint8)
    bounds = np.zeros(max(T, 1), np.int32); used = np.zeros(max(T, 1), np.int64)
    moves = np.full((2, max(n, 1)), -1, np.int32); counts = np.zeros(2, np.int32)
    rc = _load().oracle_rank_partition_tiers(n, _p(iota), _p(s), T, _p(caps), _p(prev), _p(order), _p(tier),
                                             _p(bounds), _p(used), _p(moves), _p(counts))
    if rc != 0:
        raise ValueError(f"oracle_rank_partition_tiers: bad argument (rc={rc})")
    out = dict(order=order[:n], tier=tier[:n], bounds=bounds[:T], used=used[:T])
    if prev is not None:
        # rows are n apart in the C layout
        flat = moves.reshape(-1)
        out["moves"] = [flat[k * n:k * n + counts[k]].copy() for k in range(2)]
    return out


def bfd_assign(size, iota, flags, free_pages):
    """oracle_bfd_assign -> (replica int32[m] with -1 = stays waiting, free_out int64[R])."""
    size = np.ascontiguousarray(size, dtype=np.int32)
    iota = np.ascontiguousarray(iota, dtype=np.float32)
    flags = np.ascontiguousarray(flags, dtype=np.uint8)
    free = np.ascontiguousarray(free_pages, dtype=np.int64)
    m = size.size
    assert iota.shape == (m,) and flags.shape == (m,)
    rep = np.full(max(m, 1), -9, np.int32)
    out = np.zeros(max(free.size, 1), np.int64)
    rc = _load().oracle_bfd_assign(m, _p(size), _p(iota), _p(flags), free.size, _p(free), _p(rep), _p(out))
    if rc != 0:
        raise ValueError(f"oracle_bfd_assign: bad argument (rc={rc})")
    return rep[:m].copy(), out[:free.size]


def eviction_order(which_tier, page_owner, program_tier, last_access):
    """oracle_eviction_order -> int32 array of resident pages, first to evict first."""
    owner = np.ascontiguousarray(page_owner, dtype=np.int32)
    ptier = np.ascontiguousarray(program_tier, dtype=np.uint8)
    last = np.ascontiguousarray(last_access, dtype=np.uint32)
    assert owner.shape == last.shape
    out = np.empty(max(owner.size, 1), np.int32)
    nres = C.c_int64(0)
    rc = _load().oracle_eviction_order(int(which_tier), owner.size, _p(owner), ptier.size, _p(ptier),
                                       _p(last), _p(out), C.byref(nres))
    if rc != 0:
        raise ValueError(f"oracle_eviction_order: bad argument (rc={rc})")
    return out[:nres.value].copy()


class IdlenessTracker:
    """State + the two oracle calls of Eq. (1): ``update(prog, kind, reasoning, acting)`` applies
    completed cycles (kind 0) and slot resets (kind 1) in order; ``eval(open_r, open_a)`` -> f32[n]."""

    def __init__(self, n, k=5):
        self.n, self.k = int(n), int(k)
        self.hist_r = np.zeros((self.n, self.k), np.float64)
        self.hist_a = np.zeros((self.n, self.k), np.float64)
        self.cnt = np.zeros(self.n, np.int32)

    def update(self, prog, kind, reasoning, acting):
        prog = np.ascontiguousarray(prog, dtype=np.int32)
        kind = np.ascontiguousarray(kind, dtype=np.uint8)
        r = np.ascontiguousarray(reasoning, dtype=np.float64)
        a = np.ascontiguousarray(acting, dtype=np.float64)
        assert prog.shape == kind.shape == r.shape == a.shape
        rc = _load().oracle_idleness_update(self.k, _p(self.hist_r), _p(self.hist_a), _p(self.cnt),
                                            self.n, prog.size, _p(prog), _p(kind), _p(r), _p(a))
        if rc != 0:
            raise ValueError(f"oracle_idleness_update: bad argument (rc={rc})")

    def eval(self, open_r=None, open_a=None):
        o_r = None if open_r is None else np.ascontiguousarray(open_r, dtype=np.float64)
        o_a = None if open_a is None else np.ascontiguousarray(open_a, dtype=np.float64)
        out = np.empty(self.n, np.float32)
        rc = _load().oracle_idleness_eval(self.k, _p(self.hist_r), _p(self.hist_a), _p(self.cnt),
                                          self.n, _p(o_r), _p(o_a), _p(out))
        if rc != 0:
            raise ValueError(f"oracle_idleness_eval: bad argument (rc={rc})")
        return out


def bruteforce_partition(iota, s, cap_gpu, cap_cpu):
    iota = np.ascontiguousarray(iota, dtype=np.float32)
    s = np.ascontiguousarray(s, dtype=np.int32)
    n = int(iota.shape[0])
    tier = np.zeros(max(n, 1), np.uint8)
    bounds = np.zeros(2, np.int32)
    nbest = C.c_int32(0)
    rc = _load().oracle_bruteforce_partition(n, _p(iota), _p(s), int(cap_gpu), int(cap_cpu),
                                             _p(tier), _p(bounds), C.byref(nbest))
    if rc != 0:
        raise ValueError(f"oracle_bruteforce_partition: bad argument (rc={rc})")
    return dict(tier=tier[:n], bounds=bounds, n_best=int(nbest.value))


def _move(fn, n_layers, chunk, pool, arena, a, b):
    assert pool.dtype == np.uint8 and arena.dtype == np.uint8
    assert pool.flags.c_contiguous and arena.flags.c_contiguous
    page_bytes = n_layers * chunk
    assert pool.size % page_bytes == 0 and arena.size % page_bytes == 0
    a = np.ascontiguousarray(a, dtype=np.int32)
    b = np.ascontiguousarray(b, dtype=np.int32)
    assert a.shape == b.shape
    rc = fn(n_layers, chunk, _p(pool), pool.size // page_bytes, _p(arena),
            arena.size // page_bytes, a.size, _p(a), _p(b))
    if rc != 0:
        raise ValueError(f"oracle mover: bad argument (rc={rc})")


def demote(n_layers, chunk, pool, arena, gpu_pages, host_slots):
    """pool (flat uint8 [L][P][chunk]) -> arena (flat uint8 [S][L][chunk]), in place."""
    _move(_load().oracle_demote, n_layers, chunk, pool, arena, gpu_pages, host_slots)


def promote(n_layers, chunk, pool, arena, host_slots, gpu_pages):
    _move(_load().oracle_promote, n_layers, chunk, pool, arena, host_slots, gpu_pages)


def move_slots(page_bytes, src, dst, src_slots, dst_slots):
    """src arena (flat uint8 [S1][page_bytes]) -> dst arena (flat uint8 [S2][page_bytes]), in place:
    whole page slots, one memcpy each (the arena <-> arena mover of a three-tier hierarchy)."""
    assert src.dtype == np.uint8 and dst.dtype == np.uint8 and src.flags.c_contiguous and dst.flags.c_contiguous
    assert src.size % page_bytes == 0 and dst.size % page_bytes == 0
    a = np.ascontiguousarray(src_slots, dtype=np.int32)
    b = np.ascontiguousarray(dst_slots, dtype=np.int32)
    assert a.shape == b.shape
    rc = _load().oracle_move_slots(int(page_bytes), _p(src), src.size // page_bytes, _p(dst),
                                   dst.size // page_bytes, a.size, _p(a), _p(b))
    if rc != 0:
        raise ValueError(f"oracle_move_slots: bad argument (rc={rc})")
