"""Drives the CUDA path (through the C ABI binding) over the epochs a ``workload.Sim`` plans.

Used by tests/, bench.py and __graft_entry__.smoke().  Holds the device pool, the pinned arena
and one libmori context.  No oracle here, no CPU fallback: placement comes from
``mori_rank_partition`` and bytes move through ``mori_demote`` / ``mori_promote``.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np
import torch

from . import binding
from . import workload as W


class GpuRunner:
    def __init__(self, cfg: W.Config, seed: int, path_demote=binding.PATH_AUTO,
                 path_promote=binding.PATH_AUTO, copy_kernel=binding.KERNEL_AUTO,
                 staging_bytes=0, arena: Optional[torch.Tensor] = None, device="cuda:0"):
        self.cfg, self.seed = cfg, seed
        sh = cfg.shape
        self.dev = torch.device(device)
        torch.cuda.set_device(self.dev)
        self.pool = torch.zeros(sh.n_layers * cfg.gpu_pool_pages * sh.chunk_bytes, dtype=torch.uint8,
                                device=self.dev)
        arena_bytes = cfg.cpu_pool_pages * sh.page_bytes
        if arena is None:
            arena = torch.empty(arena_bytes, dtype=torch.uint8, pin_memory=True)
        assert arena.numel() >= arena_bytes and arena.is_pinned()
        self.arena = arena[:arena_bytes]
        self.mori = binding.Mori(sh.n_layers, sh.n_kv_heads, sh.head_dim, sh.page_tokens, self.pool,
                                 self.arena, elem_bytes=sh.elem_bytes,
                                 max_programs=max(1, min(binding.MAX_PROGRAMS, cfg.n_programs)),
                                 path_demote=path_demote, path_promote=path_promote,
                                 copy_kernel=copy_kernel, staging_bytes=staging_bytes)
        self.mori_paths = (self.mori.path_demote, self.mori.path_promote)
        n = cfg.n_programs
        d = self.dev
        # device-side inputs/outputs of rank_partition + pinned mirrors for the small copies
        self.d_iota = torch.empty(n, dtype=torch.float32, device=d)
        self.d_kv = torch.empty(n, dtype=torch.int32, device=d)
        self.d_prev = torch.empty(n, dtype=torch.uint8, device=d)
        # one output blob so a single D2H brings everything back:
        #   order i32[n] | lists i32[5n] | counts i32[5] | bounds i32[2] | pad | used i64[2] | tier u8[n]
        self._o_order, self._o_lists, self._o_counts = 0, 4 * n, 4 * n + 20 * n
        self._o_bounds = self._o_counts + 20
        self._o_used = (self._o_bounds + 8 + 7) // 8 * 8
        self._o_tier = self._o_used + 16
        self.h_out = torch.zeros(self._o_tier + n, dtype=torch.uint8, pin_memory=True)
        # small n: the ranker writes its outputs straight into the pinned blob (include/mori.h:
        # outputs may be mapped host memory) -- no device-to-host copy; large n: device blob + one copy
        self.out_mapped = n <= 1024
        self.d_out = self.h_out if self.out_mapped else torch.zeros(self._o_tier + n, dtype=torch.uint8, device=d)
        self._h_out_np = self.h_out.numpy()
        self.h_in = torch.zeros(9 * n, dtype=torch.uint8, pin_memory=True)    # iota | kv | prev
        self.d_in = torch.zeros(9 * n, dtype=torch.uint8, device=d)
        self._wl = None

    # -- a1-a4 through the C ABI with HOST inputs and outputs (H2D + kernel + D2H) ---------------
    def place(self, iota: np.ndarray, kv_pages: np.ndarray, prev_tier: np.ndarray, stream=None):
        n = self.cfg.n_programs
        hin = self.h_in.numpy()
        hin[:4 * n].view(np.float32)[:] = iota
        hin[4 * n:8 * n].view(np.int32)[:] = kv_pages
        hin[8 * n:] = prev_tier
        s = stream or torch.cuda.current_stream()
        with torch.cuda.stream(s):
            self.d_in.copy_(self.h_in, non_blocking=True)
            self._launch_rank(self.d_in, s)
            if not self.out_mapped:
                self.h_out.copy_(self.d_out, non_blocking=True)
        s.synchronize()
        return self._unpack(self._h_out_np)

    # -- NEXT-1: the sticky policy mode, same host-in / host-out shape as place() ------------------
    def place_sticky(self, iota, kv_pages, prev_tier, flags, stream=None):
        n = self.cfg.n_programs
        s = stream or torch.cuda.current_stream()
        if not hasattr(self, "_st"):
            d = self.dev
            self._st = dict(flags=torch.empty(n, dtype=torch.uint8, device=d),
                            lazy=torch.empty(n, dtype=torch.uint8, device=d))
        hin = self.h_in.numpy()
        hin[:4 * n].view(np.float32)[:] = iota
        hin[4 * n:8 * n].view(np.int32)[:] = kv_pages
        hin[8 * n:] = prev_tier
        base, p = self.d_out.data_ptr(), self.d_in.data_ptr()
        with torch.cuda.stream(s):
            self.d_in.copy_(self.h_in, non_blocking=True)
            self._st["flags"].copy_(torch.from_numpy(np.ascontiguousarray(flags, dtype=np.uint8)))
            self.mori._ck(self.mori._lib.mori_sticky_rebalance(
                self.mori._h, s.cuda_stream, n, p, p + 4 * n, p + 8 * n, self._st["flags"].data_ptr(),
                self.cfg.cap_gpu_pages, self.cfg.cap_cpu_pages, base + self._o_tier,
                self._st["lazy"].data_ptr(), base + self._o_used, base + self._o_lists,
                base + self._o_counts))
            if not self.out_mapped:
                self.h_out.copy_(self.d_out, non_blocking=True)
            lazy = self._st["lazy"].cpu()
        s.synchronize()
        out = self._unpack(self._h_out_np)
        out["lazy"] = lazy.numpy()
        del out["order"], out["bounds"]
        return out

    # -- the same with the inputs already resident in HBM (bench.py 'value' leg) -------------------
    def upload_inputs(self, iota, kv_pages, prev_tier):
        n = self.cfg.n_programs
        hin = self.h_in.numpy()
        hin[:4 * n].view(np.float32)[:] = iota
        hin[4 * n:8 * n].view(np.int32)[:] = kv_pages
        hin[8 * n:] = prev_tier
        self.d_in.copy_(self.h_in, non_blocking=True)

    def place_resident(self, stream=None, done_event=None):
        """``done_event`` (a torch.cuda.Event) is recorded on the stream right behind the launch (and
        the device-to-host copy of the placement, when there is one): the device-side end of a1-a4,
        before any host-side unpacking."""
        s = stream or torch.cuda.current_stream()
        self._launch_rank(self.d_in, s)
        if not self.out_mapped:
            with torch.cuda.stream(s):
                self.h_out.copy_(self.d_out, non_blocking=True)
        if done_event is not None:
            done_event.record(s)
        s.synchronize()
        return self._unpack(self._h_out_np)

    def _launch_rank(self, d_in, s):
        n = self.cfg.n_programs
        base = self.d_out.data_ptr()
        p = d_in.data_ptr()
        self.mori._ck(self.mori._lib.mori_rank_partition(
            self.mori._h, s.cuda_stream, n, p, p + 4 * n, p + 8 * n,
            self.cfg.cap_gpu_pages, self.cfg.cap_cpu_pages,
            base + self._o_order, base + self._o_tier, base + self._o_bounds, base + self._o_used,
            base + self._o_lists, base + self._o_counts))

    def _unpack(self, buf: np.ndarray):
        n = self.cfg.n_programs
        counts = buf[self._o_counts:self._o_counts + 20].view(np.int32).copy()
        lists2d = buf[self._o_lists:self._o_lists + 20 * n].view(np.int32).reshape(5, n)
        return dict(order=buf[self._o_order:self._o_order + 4 * n].view(np.int32).copy(),
                    tier=buf[self._o_tier:self._o_tier + n].copy(),
                    bounds=buf[self._o_bounds:self._o_bounds + 8].view(np.int32).copy(),
                    used=buf[self._o_used:self._o_used + 16].view(np.int64).copy(),
                    lists=[lists2d[k, :counts[k]].copy() for k in range(5)])

    # -- a5-a7 ---------------------------------------------------------------------------------
    def prepare(self, plan: W.EpochPlan, merge=True):
        """The argument lists of the calls that will carry the epoch's moves (host work, like the
        allocator that produced the tables): ``workload.plan_calls``.  -> (steps, need_tickets)."""
        return W.plan_calls(plan, merge=merge)

    def issue(self, prepared, sync=True):
        """The C-ABI calls of one epoch, nothing else: one ``mori_demote`` / ``mori_promote`` per
        prepared step, tickets handed from the demotion that vacates pages to the promotion that
        lands in them."""
        steps, need_tickets = prepared
        lib, h_ctx = self.mori._lib, self.mori._h
        tickets = {}
        t = C.c_int64(0)
        tp = C.byref(t) if need_tickets else None
        for st in steps:
            if st[0] == "d":
                self.mori._ck(lib.mori_demote(h_ctx, st[3], st[1].ctypes.data, st[2].ctypes.data, 0, tp))
                for k in st[4]:
                    tickets[k] = t.value
            elif st[0] == "p":
                self.mori._ck(lib.mori_promote(h_ctx, st[3], st[1].ctypes.data, st[2].ctypes.data,
                                               tickets.get(st[4], 0) if st[4] > 0 else 0, 0, None))
            else:
                self.mori.mori_sync(binding.BOTH)
                tickets.clear()
        if sync:
            self.mori.mori_sync(binding.BOTH)

    def execute(self, plan: W.EpochPlan, sync=True, merge=True):
        """``prepare`` + ``issue``."""
        self.issue(self.prepare(plan, merge=merge), sync=sync)

    # -- input generation on the device (workload helper library; not the hot path) ------------
    def _keys_pages(self, triples):
        uids = np.concatenate([np.full(len(pg), uid, np.int64) for uid, first, pg in triples])
        logical = np.concatenate([first + np.arange(len(pg), dtype=np.int64) for uid, first, pg in triples])
        pages = np.concatenate([np.asarray(pg, np.int32) for uid, first, pg in triples])
        keys = W.page_keys(self.seed, uids, logical)
        return (torch.from_numpy(keys.view(np.int64)).to(self.dev),
                torch.from_numpy(pages).to(self.dev), len(pages))

    def fill(self, fills):
        """fills = [(uid, first_logical_page, gpu_pages)] -> generated content into the pool."""
        if not fills:
            return
        wl = binding.load_workload_lib()
        keys, pages, n = self._keys_pages(fills)
        sh = self.cfg.shape
        rc = wl.wl_fill_pages(self.pool.data_ptr(), self.cfg.gpu_pool_pages, sh.n_layers, sh.chunk_bytes,
                              keys.data_ptr(), pages.data_ptr(), n, 0,
                              torch.cuda.current_stream().cuda_stream)
        assert rc == 0
        torch.cuda.current_stream().synchronize()

    def check(self, triples, arena=False) -> int:
        """Mismatching 32-bit words between resident pages and the generator (device-side check;
        for ``arena`` the kernel reads the pinned arena through its mapped address)."""
        if not triples:
            return 0
        wl = binding.load_workload_lib()
        keys, pages, n = self._keys_pages(triples)
        sh = self.cfg.shape
        bad = torch.zeros(1, dtype=torch.int64, device=self.dev)
        buf = self.arena if arena else self.pool
        P = self.cfg.cpu_pool_pages if arena else self.cfg.gpu_pool_pages
        rc = wl.wl_check_pages(buf.data_ptr(), P, sh.n_layers, sh.chunk_bytes, keys.data_ptr(),
                               pages.data_ptr(), n, 1 if arena else 0, bad.data_ptr(),
                               torch.cuda.current_stream().cuda_stream)
        assert rc == 0
        return int(bad.item())

    def resident(self, sim: W.Sim):
        """(gpu triples, host triples) of every program's resident pages, for check()."""
        g, h = [], []
        for p in range(self.cfg.n_programs):
            uid = int(sim.trace.uid[p])
            if sim.gpu_pages[p].size:
                g.append((uid, 0, sim.gpu_pages[p]))
            if sim.host_slots[p].size:
                h.append((uid, 0, sim.host_slots[p]))
        return g, h

    def close(self):
        self.mori.close()


class TierRunner:
    """A three-tier hierarchy on the CUDA path (SURVEY 8f NEXT-4 ii): the paged GPU
    pool, a middle arena in device memory (a peer GPU's HBM over NVLink in production; a second
    buffer of this GPU here) and the pinned host arena.  Placement comes from
    ``mori_rank_partition_tiers``; bytes move through ``mori_demote`` / ``mori_promote`` of three
    contexts, one per pair of pools:

        pool <-> mid    the pool with a DEVICE arena (one full-grid kernel per call)
        pool <-> host   the hot path's context (staged / zero-copy over the host link)
        mid  <-> host   the middle arena described as a pool of ONE layer whose chunk is a whole
                        page (n_kv_heads = L * H): a slot is then one contiguous chunk, and the
                        arena <-> arena move is the same gather -> staging -> DMA pipeline

    ``workload.SimTiers`` never reuses an id freed in the current phase before a join, so the three
    contexts need no tickets between them."""

    def __init__(self, cfg: W.Config, seed: int, mid_slots: int, host_arena: Optional[torch.Tensor] = None,
                 staging_bytes=0, device="cuda:0"):
        self.cfg, self.seed = cfg, seed
        sh = cfg.shape
        self.dev = torch.device(device)
        torch.cuda.set_device(self.dev)
        self.pool = torch.zeros(sh.n_layers * cfg.gpu_pool_pages * sh.chunk_bytes, dtype=torch.uint8, device=self.dev)
        self.mid = torch.zeros(mid_slots * sh.page_bytes, dtype=torch.uint8, device=self.dev)
        host_bytes = cfg.cpu_pool_pages * sh.page_bytes
        if host_arena is None:
            host_arena = torch.empty(host_bytes, dtype=torch.uint8, pin_memory=True)
        self.host = host_arena[:host_bytes]
        n = max(1, min(binding.MAX_PROGRAMS, cfg.n_programs))
        kw = dict(elem_bytes=sh.elem_bytes, max_programs=n, staging_bytes=staging_bytes)
        self.pool_mid = binding.Mori(sh.n_layers, sh.n_kv_heads, sh.head_dim, sh.page_tokens, self.pool, self.mid, **kw)
        self.pool_host = binding.Mori(sh.n_layers, sh.n_kv_heads, sh.head_dim, sh.page_tokens, self.pool, self.host, **kw)
        self.mid_host = binding.Mori(1, sh.n_layers * sh.n_kv_heads, sh.head_dim, sh.page_tokens, self.mid, self.host, **kw)
        assert self.mid_host.chunk_bytes == sh.page_bytes
        self.ctxs = (self.pool_mid, self.pool_host, self.mid_host)
        d = self.dev
        self.n = cfg.n_programs
        self.d_iota = torch.empty(self.n, dtype=torch.float32, device=d)
        self.d_kv = torch.empty(self.n, dtype=torch.int32, device=d)
        self.d_prev = torch.empty(self.n, dtype=torch.uint8, device=d)
        self.d_order = torch.empty(self.n, dtype=torch.int32, device=d)
        self.d_tier = torch.empty(self.n, dtype=torch.uint8, device=d)
        self.d_bounds = torch.empty(3, dtype=torch.int32, device=d)
        self.d_used = torch.empty(3, dtype=torch.int64, device=d)
        self.d_moves = torch.empty(2 * self.n, dtype=torch.int32, device=d)
        self.d_counts = torch.empty(2, dtype=torch.int32, device=d)

    def place(self, iota, kv_pages, prev_tier, caps):
        n = self.n
        self.d_iota.copy_(torch.from_numpy(np.ascontiguousarray(iota, dtype=np.float32)))
        self.d_kv.copy_(torch.from_numpy(np.ascontiguousarray(kv_pages, dtype=np.int32)))
        self.d_prev.copy_(torch.from_numpy(np.ascontiguousarray(prev_tier, dtype=np.uint8)))
        self.pool_host.mori_rank_partition_tiers(n, self.d_iota, self.d_kv, caps, self.d_order, self.d_tier,
                                                 self.d_bounds, self.d_used, prev_tier=self.d_prev,
                                                 moves=self.d_moves, move_counts=self.d_counts)
        torch.cuda.synchronize()
        c, mv = self.d_counts.cpu().numpy(), self.d_moves.cpu().numpy()
        return dict(order=self.d_order.cpu().numpy(), tier=self.d_tier.cpu().numpy(), bounds=self.d_bounds.cpu().numpy(),
                    used=self.d_used.cpu().numpy(), moves=[mv[k * n:k * n + c[k]].copy() for k in range(2)])

    def execute(self, plan: W.EpochPlan):
        """One flat call per (from, to) pair and phase; a join where the planner asks for one."""
        batch = {}

        def flush():
            for (frm, to), ops in batch.items():
                src = np.concatenate([o[4] for o in ops])
                dst = np.concatenate([o[5] for o in ops])
                lo, hi = min(frm, to), max(frm, to)
                ctx = {(0, 1): self.pool_mid, (0, 2): self.pool_host, (1, 2): self.mid_host}[(lo, hi)]
                if to > frm:
                    ctx.mori_demote(src, dst)                 # faster tier's ids first
                else:
                    ctx.mori_promote(src, dst)                # (slower tier's slots, faster tier's ids)
            batch.clear()

        def join():
            for c in self.ctxs:
                c.mori_sync(binding.BOTH)

        for op in plan.ops:
            if op[0] == "move":
                batch.setdefault((op[2], op[3]), []).append(op)
            elif op[0] == "sync_all":
                flush(); join()
        flush(); join()

    def fill(self, fills):
        if not fills:
            return
        wl = binding.load_workload_lib()
        keys, pages, n = self._keys_pages(fills)
        sh = self.cfg.shape
        rc = wl.wl_fill_pages(self.pool.data_ptr(), self.cfg.gpu_pool_pages, sh.n_layers, sh.chunk_bytes,
                              keys.data_ptr(), pages.data_ptr(), n, 0, torch.cuda.current_stream().cuda_stream)
        assert rc == 0
        torch.cuda.current_stream().synchronize()

    _keys_pages = GpuRunner._keys_pages

    def close(self):
        for c in self.ctxs:
            c.close()
