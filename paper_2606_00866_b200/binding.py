"""ctypes binding over libmori.so -- argument marshalling only; every step runs in the library.

Function names mirror include/mori.h.  Tensors are passed as ``data_ptr()``; torch is used for
device memory and streams and nowhere else.  There is NO fallback: if the CUDA library cannot be
loaded this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmori.so")
WORKLOAD_LIB_PATH = os.path.join(_HERE, "libmori_workload.so")

OK, ERR_INVALID_ARG, ERR_CUDA, ERR_CAPACITY, ERR_STATE, ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
TIER_GPU, TIER_CPU, TIER_WAIT = 0, 1, 2
DEMOTE, PROMOTE, BOTH = 1, 2, 3
PATH_AUTO, PATH_ZEROCOPY, PATH_STAGED, PATH_COPYENGINE = 0, 1, 2, 3
KERNEL_AUTO, KERNEL_LDST, KERNEL_TMA = 0, 1, 2
MAX_PROGRAMS = 8192
FLAG_ACTING, FLAG_READY, FLAG_NEW = 1, 2, 4
PATH_NAMES = {1: "zerocopy", 2: "staged", 3: "copyengine"}
KERNEL_NAMES = {1: "ldst", 2: "tma"}

EXPORTS = ["mori_create", "mori_destroy", "mori_rank_partition", "mori_demote", "mori_promote",
           "mori_sync", "mori_after_stream", "mori_stream_wait", "mori_gather_pages",
           "mori_scatter_pages", "mori_profile", "mori_profile_read", "mori_path",
           "mori_copy_kernel", "mori_last_error", "mori_launch_count", "mori_host_alloc",
           "mori_host_free", "mori_sticky_rebalance", "mori_idleness_update",
           "mori_idleness_eval", "mori_eviction_order", "mori_bfd_assign",
           "mori_rank_partition_tiers", "mori_profile_timeline", "mori_noop", "mori_eviction_order_noalloc"]


class MoriConfig(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("page_tokens", C.c_int32), ("elem_bytes", C.c_int32),
                ("gpu_pool", C.c_void_p), ("gpu_pool_pages", C.c_int64),
                ("host_arena", C.c_void_p), ("host_arena_slots", C.c_int64),
                ("max_programs", C.c_int32), ("path_demote", C.c_int32),
                ("path_promote", C.c_int32), ("copy_kernel", C.c_int32),
                ("staging_bytes", C.c_int64), ("max_pages_per_call", C.c_int64),
                ("zerocopy_ctas", C.c_int32), ("idleness_window", C.c_int32)]


class MoriError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"mori status {code}: {msg}")
        self.code = code


_lib = None


def load():
    """Loads libmori.so (built in-tree by ``paper_2606_00866_b200.build``).  Raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_00866_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.mori_create.argtypes = [C.POINTER(MoriConfig), C.POINTER(vp)]
        L.mori_destroy.argtypes = [vp]
        L.mori_rank_partition.argtypes = [vp, vp, i32, vp, vp, vp, i64, i64, vp, vp, vp, vp, vp, vp]
        L.mori_sticky_rebalance.argtypes = [vp, vp, i32, vp, vp, vp, vp, i64, i64, vp, vp, vp, vp, vp]
        L.mori_rank_partition_tiers.argtypes = [vp, vp, i32, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp]
        L.mori_bfd_assign.argtypes = [vp, vp, i32, vp, vp, vp, i32, vp, vp, vp]
        L.mori_eviction_order.argtypes = [vp, vp, i32, i64, vp, i32, vp, vp, vp, vp]
        L.mori_idleness_update.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        L.mori_idleness_eval.argtypes = [vp, vp, i32, vp, vp, vp]
        L.mori_demote.argtypes = [vp, i64, vp, vp, i64, vp]
        L.mori_promote.argtypes = [vp, i64, vp, vp, i64, i64, vp]
        L.mori_sync.argtypes = [vp, i32]
        L.mori_after_stream.argtypes = [vp, i32, vp]
        L.mori_stream_wait.argtypes = [vp, vp, i32]
        L.mori_gather_pages.argtypes = [vp, vp, i64, vp, vp]
        L.mori_scatter_pages.argtypes = [vp, vp, i64, vp, vp]
        L.mori_profile.argtypes = [vp, i32]
        L.mori_profile_read.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(i64), C.POINTER(i64)]
        L.mori_profile_timeline.argtypes = [vp, i32, i64, vp, vp, vp, vp, C.POINTER(i64)]
        L.mori_noop.argtypes = [vp, vp]
        L.mori_eviction_order_noalloc.argtypes = [vp, i32, i64, vp, i32, vp, vp, vp, vp, C.POINTER(C.c_char_p)]
        L.mori_path.argtypes = [vp, i32]
        L.mori_copy_kernel.argtypes = [vp]
        L.mori_last_error.argtypes = [vp]
        L.mori_launch_count.argtypes = [vp, C.POINTER(i64)]
        L.mori_host_alloc.argtypes = [i64, C.POINTER(vp)]
        L.mori_host_free.argtypes = [vp]
        L.mori_last_error.restype = C.c_char_p
        for name in EXPORTS:
            if name != "mori_last_error":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _ptr(t) -> Optional[int]:
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream_handle(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _host_i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


class Mori:
    """One libmori context.  ``gpu_pool`` is a CUDA uint8/bf16 tensor of the whole pool,
    ``host_arena`` a pinned CPU tensor (or None for rank/partition and device gather only)."""

    def __init__(self, n_layers, n_kv_heads, head_dim, page_tokens, gpu_pool, host_arena=None,
                 elem_bytes=2, max_programs=MAX_PROGRAMS, path_demote=PATH_AUTO,
                 path_promote=PATH_AUTO, copy_kernel=KERNEL_AUTO, staging_bytes=0,
                 max_pages_per_call=0, zerocopy_ctas=0, idleness_window=0):
        self._lib = load()
        self.chunk_bytes = 2 * n_kv_heads * page_tokens * head_dim * elem_bytes
        self.page_bytes = self.chunk_bytes * n_layers
        self.n_layers = n_layers
        pool_bytes = gpu_pool.numel() * gpu_pool.element_size()
        assert gpu_pool.is_cuda and gpu_pool.is_contiguous() and pool_bytes % self.page_bytes == 0
        self.gpu_pool, self.host_arena = gpu_pool, host_arena      # keep alive
        self.gpu_pool_pages = pool_bytes // self.page_bytes
        cfg = MoriConfig(n_layers, n_kv_heads, head_dim, page_tokens, elem_bytes,
                         gpu_pool.data_ptr(), self.gpu_pool_pages, None, 0, max_programs,
                         path_demote, path_promote, copy_kernel, staging_bytes, max_pages_per_call,
                         zerocopy_ctas, idleness_window)
        self.host_arena_slots = 0
        if host_arena is not None:
            arena_bytes = host_arena.numel() * host_arena.element_size()
            assert (host_arena.is_cuda or host_arena.is_pinned()) and host_arena.is_contiguous()
            assert arena_bytes % self.page_bytes == 0
            self.host_arena_slots = arena_bytes // self.page_bytes
            cfg.host_arena, cfg.host_arena_slots = host_arena.data_ptr(), self.host_arena_slots
        h = C.c_void_p()
        rc = self._lib.mori_create(C.byref(cfg), C.byref(h))
        if rc != OK:
            raise MoriError(rc, (self._lib.mori_last_error(None) or b"").decode())
        self._h = h

    # -- plumbing ----------------------------------------------------------------------------
    def _ck(self, rc: int) -> int:
        if rc != OK:
            raise MoriError(rc, (self._lib.mori_last_error(self._h) or b"").decode())
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self._lib.mori_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def mori_path(self, which) -> int:
        return self._lib.mori_path(self._h, which)

    def mori_copy_kernel(self) -> int:
        return self._lib.mori_copy_kernel(self._h)

    @property
    def path_demote(self) -> int:
        return self.mori_path(DEMOTE)

    @property
    def path_promote(self) -> int:
        return self.mori_path(PROMOTE)

    @property
    def copy_kernel(self) -> int:
        return self.mori_copy_kernel()

    # -- a1-a4 -------------------------------------------------------------------------------
    def mori_rank_partition(self, n, idleness, kv_pages, prev_tier, gpu_cap_pages, cpu_cap_pages,
                            order, tier, bounds, used_pages, lists=None, list_counts=None,
                            stream=None):
        """All array arguments are CUDA tensors (see include/mori.h); asynchronous on ``stream``."""
        return self._ck(self._lib.mori_rank_partition(
            self._h, _stream_handle(stream), int(n), _ptr(idleness), _ptr(kv_pages), _ptr(prev_tier),
            int(gpu_cap_pages), int(cpu_cap_pages), _ptr(order), _ptr(tier), _ptr(bounds),
            _ptr(used_pages), _ptr(lists), _ptr(list_counts)))

    # -- NEXT-1: sticky, status-aware tier management ----------------------------------------
    def mori_sticky_rebalance(self, n, idleness, kv_pages, prev_tier, flags, gpu_cap_pages,
                              cpu_cap_pages, tier, lazy, used_pages, lists, list_counts, stream=None):
        """All array arguments are CUDA tensors (see include/mori.h); asynchronous on ``stream``."""
        return self._ck(self._lib.mori_sticky_rebalance(
            self._h, _stream_handle(stream), int(n), _ptr(idleness), _ptr(kv_pages), _ptr(prev_tier),
            _ptr(flags), int(gpu_cap_pages), int(cpu_cap_pages), _ptr(tier), _ptr(lazy),
            _ptr(used_pages), _ptr(lists), _ptr(list_counts)))

    # -- NEXT-4(ii): the partition with T capacities --------------------------------------------
    def mori_rank_partition_tiers(self, n, idleness, kv_pages, cap_pages, order, tier, bounds,
                                  used_pages, prev_tier=None, moves=None, move_counts=None, stream=None):
        """``cap_pages``: host sequence of 1..8 capacities; the rest are CUDA tensors."""
        caps = np.ascontiguousarray(cap_pages, dtype=np.int64)
        return self._ck(self._lib.mori_rank_partition_tiers(
            self._h, _stream_handle(stream), int(n), _ptr(idleness), _ptr(kv_pages), int(caps.size),
            caps.ctypes.data, _ptr(prev_tier), _ptr(order), _ptr(tier), _ptr(bounds), _ptr(used_pages),
            _ptr(moves), _ptr(move_counts)))

    # -- NEXT-4(i): Best-Fit-Decreasing across replicas ------------------------------------------
    def mori_bfd_assign(self, size, idleness, flags, free_pages, replica, free_out, stream=None):
        """CUDA tensors int32[m], float32[m], uint8[m], int64[R]; outputs int32[m], int64[R]."""
        return self._ck(self._lib.mori_bfd_assign(
            self._h, _stream_handle(stream), int(size.numel()), _ptr(size), _ptr(idleness), _ptr(flags),
            int(free_pages.numel()), _ptr(free_pages), _ptr(replica), _ptr(free_out)))

    # -- NEXT-3: typed eviction order -----------------------------------------------------------
    def mori_eviction_order(self, which_tier, page_owner, program_tier, last_access, victims,
                            n_resident, stream=None):
        """CUDA tensors: int32[n_pages], uint8[n_programs], uint32-as-int32[n_pages]; outputs
        int32[n_pages], int32[1]."""
        return self._ck(self._lib.mori_eviction_order(
            self._h, _stream_handle(stream), int(which_tier), int(page_owner.numel()), _ptr(page_owner),
            int(program_tier.numel()), _ptr(program_tier), _ptr(last_access), _ptr(victims),
            _ptr(n_resident)))

    NOALLOC_MAX_PAGES = 65536

    @staticmethod
    def mori_eviction_order_noalloc(which_tier, page_owner, program_tier, last_access, victims, n_resident,
                                    stream=None):
        """The typed eviction order with NO allocation on any call and no context: the sort scratch
        is a 1 MiB static device array (include/mori.h).  At most ``NOALLOC_MAX_PAGES`` pages; calls
        that overlap on the GPU race on the shared scratch.  Same tensors as ``mori_eviction_order``."""
        why = C.c_char_p()
        rc = load().mori_eviction_order_noalloc(
            _stream_handle(stream), int(which_tier), int(page_owner.numel()), _ptr(page_owner),
            int(program_tier.numel()), _ptr(program_tier), _ptr(last_access), _ptr(victims), _ptr(n_resident),
            C.byref(why))
        if rc != OK:
            raise MoriError(rc, (why.value or b"").decode())
        return rc

    # -- NEXT-2: Eq. (1) on the device -------------------------------------------------------
    def mori_idleness_update(self, prog, kind, reasoning, acting, stream=None):
        """CUDA tensors int32[m], uint8[m], float64[m], float64[m]; applied in list order."""
        return self._ck(self._lib.mori_idleness_update(
            self._h, _stream_handle(stream), int(prog.numel()), _ptr(prog), _ptr(kind), _ptr(reasoning),
            _ptr(acting)))

    def mori_idleness_eval(self, n, open_reasoning, open_acting, idleness_out, stream=None):
        return self._ck(self._lib.mori_idleness_eval(
            self._h, _stream_handle(stream), int(n), _ptr(open_reasoning), _ptr(open_acting),
            _ptr(idleness_out)))

    # -- a5-a7 -------------------------------------------------------------------------------
    def mori_demote(self, gpu_pages, host_slots, wait_promote_ticket=0, want_ticket=True) -> int:
        """-> the call's ticket (0 with ``want_ticket=False``: ticket_out = NULL, no event is recorded)."""
        g, h = _host_i32(gpu_pages), _host_i32(host_slots)
        assert g.shape == h.shape and g.ndim == 1
        t = C.c_int64(0)
        self._ck(self._lib.mori_demote(self._h, g.size, g.ctypes.data, h.ctypes.data,
                                       int(wait_promote_ticket), C.byref(t) if want_ticket else None))
        return t.value

    def mori_promote(self, host_slots, gpu_pages, pages_after_demote=0, slots_after_demote=0,
                     want_ticket=True) -> int:
        g, h = _host_i32(gpu_pages), _host_i32(host_slots)
        assert g.shape == h.shape and g.ndim == 1
        t = C.c_int64(0)
        self._ck(self._lib.mori_promote(self._h, g.size, h.ctypes.data, g.ctypes.data,
                                        int(pages_after_demote), int(slots_after_demote),
                                        C.byref(t) if want_ticket else None))
        return t.value

    def mori_sync(self, which=BOTH):
        return self._ck(self._lib.mori_sync(self._h, which))

    def mori_after_stream(self, which=BOTH, stream=None):
        return self._ck(self._lib.mori_after_stream(self._h, which, _stream_handle(stream)))

    def mori_stream_wait(self, stream=None, which=BOTH):
        return self._ck(self._lib.mori_stream_wait(self._h, _stream_handle(stream), which))

    # -- device halves -----------------------------------------------------------------------
    def mori_gather_pages(self, gpu_pages_dev, dst, stream=None):
        return self._ck(self._lib.mori_gather_pages(self._h, _stream_handle(stream),
                                                    gpu_pages_dev.numel(), _ptr(gpu_pages_dev), _ptr(dst)))

    def mori_scatter_pages(self, gpu_pages_dev, src, stream=None):
        return self._ck(self._lib.mori_scatter_pages(self._h, _stream_handle(stream),
                                                     gpu_pages_dev.numel(), _ptr(gpu_pages_dev), _ptr(src)))

    # -- pinned host memory ------------------------------------------------------------------
    @staticmethod
    def mori_host_alloc(nbytes: int):
        """-> uint8 torch tensor over ``nbytes`` of pinned, device-mapped host memory (exact size,
        unlike torch's pinned allocator which rounds up to a power of two).  Free it with
        ``mori_host_free(t)`` after closing every context that uses it."""
        import torch
        torch.cuda.init()            # is_pinned() answers False before torch's lazy CUDA init
        lib = load()
        p = C.c_void_p()
        rc = lib.mori_host_alloc(int(nbytes), C.byref(p))
        if rc != OK:
            raise MoriError(rc, (lib.mori_last_error(None) or b"").decode())
        t = torch.frombuffer((C.c_uint8 * int(nbytes)).from_address(p.value), dtype=torch.uint8)
        t._mori_host_ptr = p.value
        return t

    @staticmethod
    def mori_host_free(t):
        p = getattr(t, "_mori_host_ptr", None)
        if p:
            t._mori_host_ptr = None
            return load().mori_host_free(p)
        return OK

    def mori_noop(self, stream=None):
        return self._ck(self._lib.mori_noop(self._h, _stream_handle(stream)))

    # -- profiling ---------------------------------------------------------------------------
    def mori_launch_count(self) -> int:
        n = C.c_int64(0)
        self._ck(self._lib.mori_launch_count(self._h, C.byref(n)))
        return n.value

    def mori_profile(self, enable):
        """False / True, or 2 to keep a timeline as well (``mori_profile_timeline``)."""
        return self._ck(self._lib.mori_profile(self._h, int(enable)))

    def mori_profile_timeline(self, which):
        """-> list of (kind, start_ms, end_ms, bytes): kind 0 = kernel, 1 = a segment's DMAs."""
        n = C.c_int64(0)
        self._ck(self._lib.mori_profile_timeline(self._h, which, 0, None, None, None, None, C.byref(n)))
        k = np.zeros(n.value, np.int32); t0 = np.zeros(n.value); t1 = np.zeros(n.value); b = np.zeros(n.value, np.int64)
        self._ck(self._lib.mori_profile_timeline(self._h, which, n.value, k.ctypes.data, t0.ctypes.data,
                                                 t1.ctypes.data, b.ctypes.data, C.byref(n)))
        return [(int(k[i]), float(t0[i]), float(t1[i]), int(b[i])) for i in range(n.value)]

    def mori_profile_read(self, which):
        ms, n, b = C.c_double(0), C.c_int64(0), C.c_int64(0)
        self._ck(self._lib.mori_profile_read(self._h, which, C.byref(ms), C.byref(n), C.byref(b)))
        return ms.value, n.value, b.value


# ------------------------------------------------------------------------------------------------
# workload helper library (input generation on the device; not part of the hot path)
# ------------------------------------------------------------------------------------------------
_wl = None


def load_workload_lib():
    global _wl
    if _wl is None:
        if not os.path.exists(WORKLOAD_LIB_PATH):
            raise RuntimeError(f"{WORKLOAD_LIB_PATH} is missing: run `python -m paper_2606_00866_b200.build`")
        L = C.CDLL(WORKLOAD_LIB_PATH)
        vp = C.c_void_p
        L.wl_fill_pages.argtypes = [vp, C.c_longlong, C.c_int, C.c_int, vp, vp, C.c_longlong, C.c_int, vp]
        L.wl_check_pages.argtypes = [vp, C.c_longlong, C.c_int, C.c_int, vp, vp, C.c_longlong, C.c_int, vp, vp]
        L.wl_fill_pages.restype = C.c_int
        L.wl_check_pages.restype = C.c_int
        _wl = L
    return _wl
