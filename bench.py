#!/usr/bin/env python
"""bench.py -- the MORI hot path on B200, measured (driver contract: one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--f-busy F] [--impl ours|reference]
    python bench.py --leg copy_sweep          (auxiliary: the gather/scatter kernel alone and in-step)

A *step* is one scheduling epoch: every row of SURVEY.md section 8(a) once --
``mori_rank_partition`` (a1-a4), ``mori_demote`` / ``mori_promote`` for every program the placement
moves (a5, a6, concurrently in both link directions) and ``mori_sync`` (a7) -- on the seeded
synthetic workload of BASELINE.json ``configs[1]`` (cfg 2, Llama-3-8B-shaped KV, 64 programs,
60 GiB device pool, 128 GiB pinned arena).  Everything on the path runs in
libmori.so (CUDA, sm_100a) through its C ABI; there is no CPU fallback.  After the headline config
a single-GPU run measures every other BASELINE.json config the same way (``per_config``).

Numbers on the line (DESIGN.md section 7 says how each is derived):
  value        migrated KV bytes / time of K epochs, GB/s.  The KV pool and the rank/partition
               inputs are resident in HBM when the timed region starts; timed on the device with
               CUDA events (region A: rank/partition up to the arrival of its move lists in host
               memory, region B: all demotes/promotes up to the join).  The page/slot allocator
               between A and B, and the concatenation of its tables into the calls' arguments, are
               harness code (they stand in for the serving engine's allocator) and are not timed.
  frac_of_measured_link_peak, roofline_frac   the two headline fractions, right behind ``value``.
  e2e          the same epochs' metric through the public API from HOST buffers: idleness / size /
               previous-tier arrays copied host->device, lists device->host, host page tables
               into mori_demote / mori_promote, the allocator included, one timed region.
  roofline     the gather/scatter kernel of the STAGED path (the only HBM-bound kernel), timed
               live by the library's CUDA events around every launch inside the timed steps.
  per_config   one record per BASELINE.json config: GB/s, fraction of the measured link peak, scale,
               the ranker's capacities, in-step and standalone gather/scatter fractions.
  link         measured pinned-memcpy peaks of this box (denominators) and the achieved fractions.
  gather_scatter  the device halves alone (pool <-> contiguous device buffer), >= 4 GiB per launch.
  rank_partition, eviction_order   the latency-bound entry points against the launch floor (mori_noop).
  cpu_baseline the CPU oracle (oracle/, as it stands) on this box's host cores, 1 thread and all
               cores, bounded sample, on the scaled twin of every config.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "kv_migration_GBps"
UNIT = "GB/s"
SEED = 866
GIB = 1 << 30


# ------------------------------------------------------------------------------------------------
# helpers
# ------------------------------------------------------------------------------------------------
def _meminfo_kb(key: str) -> int:
    with open("/proc/meminfo") as f:
        for line in f:
            if line.startswith(key + ":"):
                return int(line.split()[1])
    return 0


class ClockSampler:
    """nvidia-smi clocks + throttle reasons every 200 ms while the timed region runs
    (B200_PROFILING.md 'clocks line')."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for k, name in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measure_link_peak(arena, nbytes=GIB, reps=5, stream_chunks=1, joined=False):
    """Pinned cudaMemcpyAsync of ONE contiguous buffer: D2H alone, H2D alone, both at once on
    two streams -- the host-link denominators (GB/s).  Uses the first bytes of the arena before
    the workload touches it, and a scratch device buffer."""
    import torch
    nbytes = min(nbytes, arena.numel() // 2)
    nbytes -= nbytes % 4096
    h1, h2 = arena[:nbytes], arena[nbytes:2 * nbytes]
    d1 = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    d2 = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def run(do_d2h, do_h2d):
        best = float("inf")
        for _ in range(reps):
            torch.cuda.synchronize()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            cur = torch.cuda.current_stream()
            e0 = torch.cuda.Event(enable_timing=True); e0.record(cur)
            if do_d2h and do_h2d:
                s1.wait_event(e0); s2.wait_event(e0)
                with torch.cuda.stream(s1):
                    h1.copy_(d1, non_blocking=True)
                with torch.cuda.stream(s2):
                    d2.copy_(h2, non_blocking=True)
                cur.wait_stream(s1); cur.wait_stream(s2)
            elif joined:                                 # one direction, issued the way an epoch's transfers are:
                s1.wait_event(e0)                        # on a side stream, joined to the timing stream on both ends
                with torch.cuda.stream(s1):
                    if do_d2h:
                        h1.copy_(d1, non_blocking=True)
                    else:
                        d2.copy_(h2, non_blocking=True)
                cur.wait_stream(s1)
            elif do_d2h:                                 # one direction: the copy alone between the two events
                h1.copy_(d1, non_blocking=True)
            else:
                d2.copy_(h2, non_blocking=True)
            e1 = torch.cuda.Event(enable_timing=True); e1.record(cur)
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
            del ev
        return best * 1e-3

    out = {"bytes": nbytes,
           "d2h": nbytes / run(True, False) / 1e9,
           "h2d": nbytes / run(False, True) / 1e9,
           "bidir_sum": 2 * nbytes / run(True, True) / 1e9}
    if stream_chunks > 1:
        # the same copy streamed over `stream_chunks` successive regions of the arena, ONE timing:
        # what the link sustains right now (on a box that has been busy for minutes this reads a
        # few per cent under the best-of-5 figure above; on a fresh box the two agree)
        k = int(min(stream_chunks, arena.numel() // nbytes))
        for name, d2h in (("d2h_streamed", True), ("h2d_streamed", False)):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(s1)
            with torch.cuda.stream(s1):
                for i in range(k):
                    h = arena[i * nbytes:(i + 1) * nbytes]
                    if d2h:
                        h.copy_(d1, non_blocking=True)
                    else:
                        d1.copy_(h, non_blocking=True)
            e1.record(s1)
            torch.cuda.synchronize()
            out[name] = k * nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9
        out["streamed_chunks"] = k
    del d1, d2
    return out


def ideal_seconds(dem_bytes, pro_bytes, link):
    """Lower bound on an epoch's transfer time from the measured pinned-memcpy peaks."""
    return max(dem_bytes / (link["d2h"] * 1e9), pro_bytes / (link["h2d"] * 1e9),
               (dem_bytes + pro_bytes) / (link["bidir_sum"] * 1e9))


def memcpy_model_seconds(dem_bytes, pro_bytes, link):
    """Time two plain pinned memcpys of these sizes, started together, would take at the measured
    rates: both directions share the link at the measured simultaneous rate (split in
    proportion to the solo rates) until the shorter one ends, the rest runs at its solo rate.
    Tighter than ``ideal_seconds`` when the two directions carry different amounts."""
    d_solo, p_solo = link["d2h"] * 1e9, link["h2d"] * 1e9
    both = link["bidir_sum"] * 1e9
    d_both, p_both = both * d_solo / (d_solo + p_solo), both * p_solo / (d_solo + p_solo)
    if dem_bytes == 0 or pro_bytes == 0:
        return dem_bytes / d_solo + pro_bytes / p_solo
    t = min(dem_bytes / d_both, pro_bytes / p_both)
    return t + (dem_bytes - t * d_both) / d_solo + (pro_bytes - t * p_both) / p_solo


# ------------------------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline, --impl reference): the only places bench.py touches oracle/
# ------------------------------------------------------------------------------------------------
def _cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


class OracleEpochs:
    """The oracle as it stands on a scaled twin of a bench workload (same L/H/D/T/n, pools and
    contexts divided by ``scale`` so that byte mirrors of both pools fit host RAM).  ``threads``
    > 1 splits the pages of every move evenly over that many host threads, each calling the
    oracle's single-threaded mover on its share (the threading lives here, not in oracle.c; ctypes
    releases the GIL for the duration of a call)."""

    def __init__(self, cfg_index: int, scale: int, seed: int, f_busy=None):
        import oracle
        from paper_2606_00866_b200 import workload as W
        self.oracle, self.W = oracle, W
        oracle.build()
        self.cfg = W.get_config(cfg_index, scale, f_busy)
        sh = self.cfg.shape
        self.sim = W.Sim(self.cfg, seed)
        # byte mirrors of both pools; contents are irrelevant to the timing, every page is touched
        self.pool = np.empty(sh.n_layers * self.cfg.gpu_pool_pages * sh.chunk_bytes, np.uint8)
        self.arena = np.empty(self.cfg.cpu_pool_pages * sh.page_bytes, np.uint8)
        self._touch(self.pool, 0x5A)
        self._touch(self.arena, 0x01)
        self.pool_exec = None

    @staticmethod
    def _touch(a, v):
        from concurrent.futures import ThreadPoolExecutor
        n = max(1, min(os.cpu_count() or 1, 8))
        step = -(-a.size // n)
        with ThreadPoolExecutor(n) as ex:
            list(ex.map(lambda k: a[k * step:(k + 1) * step:4096].fill(v), range(n)))

    def _move(self, fn, a, b, threads):
        sh = self.cfg.shape
        if threads <= 1 or len(a) < 2 * threads:
            fn(sh.n_layers, sh.chunk_bytes, self.pool, self.arena, a, b)
            return
        if self.pool_exec is None or self.pool_exec._max_workers != threads:
            from concurrent.futures import ThreadPoolExecutor
            self.pool_exec = ThreadPoolExecutor(threads)
        cuts = np.linspace(0, len(a), threads + 1).astype(int)
        futs = [self.pool_exec.submit(fn, sh.n_layers, sh.chunk_bytes, self.pool, self.arena,
                                      a[cuts[t]:cuts[t + 1]], b[cuts[t]:cuts[t + 1]]) for t in range(threads)]
        for f in futs:
            f.result()

    def step(self, threads=1):
        """One epoch.  -> (seconds in the oracle, bytes migrated)."""
        cfg, sh, o = self.cfg, self.cfg.shape, self.oracle
        plan = self.sim.begin_epoch()
        t0 = time.perf_counter()
        res = o.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        t = time.perf_counter() - t0
        self.sim.apply_placement(res["tier"], res["lists"])
        t0 = time.perf_counter()
        for op in plan.ops:
            if op[0] == "demote":
                self._move(o.demote, op[3], op[4], threads)
            elif op[0] == "promote":
                self._move(o.promote, op[3], op[4], threads)
        t += time.perf_counter() - t0
        self.sim.end_epoch()                         # page contents are irrelevant to the timing
        return t, (plan.demote_pages + plan.promote_pages) * sh.page_bytes


def cpu_baseline(cfg_index: int, budget_s: float = 6.0, scale: int = 16, f_busy=None, max_bytes=12 * GIB):
    """The oracle as it stands on the box's host cores: one thread, then all cores (pages of every
    move split evenly), on alternating epochs of the scaled twin of config ``cfg_index``."""
    from paper_2606_00866_b200 import workload as W
    while True:                                      # mirrors of both pools must stay small enough to touch quickly
        c = W.get_config(cfg_index, scale, f_busy)
        if (c.gpu_pool_pages + c.cpu_pool_pages) * c.shape.page_bytes <= max_bytes or c.cpu_pool_pages < 64:
            break
        scale *= 2
    oe = OracleEpochs(cfg_index, scale, SEED, f_busy)
    cores = os.cpu_count() or 1
    for _ in range(3):
        oe.step()
    acc = {1: [0.0, 0, 0], cores: [0.0, 0, 0]}
    t_wall, n = time.perf_counter(), 0
    while (time.perf_counter() - t_wall < budget_s and n < oe.cfg.epochs - 3) or n < 4:
        th = 1 if n % 2 == 0 else cores
        t, b = oe.step(th)
        acc[th][0] += t; acc[th][1] += b; acc[th][2] += 1
        n += 1
    def gbps(a):
        return a[1] / a[0] / 1e9 if a[0] > 0 and a[1] > 0 else 0.0
    sample = (f"{n} epochs of {oe.cfg.name} (cfg {cfg_index} with pools and contexts / {scale}, same L/H/D/T/n), "
              f"alternating 1 thread / {cores} threads; {acc[1][1] / GIB:.1f} + {acc[cores][1] / GIB:.1f} GiB migrated "
              f"host->host by oracle.c (qsort + prefix loop + per-(page,layer) memcpy; threads split a move's pages evenly)")
    return {"value": gbps(acc[1]), "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
            "all_cores": {"value": gbps(acc[cores]), "unit": UNIT, "cores": cores},
            "host_cores_available": cores, "cpu_model": _cpu_model(), "scale": scale, "workload": oe.cfg.name}


def _reference_scale(cfg_index: int, W, f_busy=None) -> int:
    """The smallest power-of-two scale whose byte mirrors of BOTH pools fit this host (80 % of
    MemAvailable): /2 for cfg 2 on a 196 GiB box."""
    avail = int(_meminfo_kb("MemAvailable") * 1024 * 0.80)
    scale = 1
    while True:
        c = W.get_config(cfg_index, scale, f_busy)
        if (c.gpu_pool_pages + c.cpu_pool_pages) * c.shape.page_bytes <= avail:
            return scale
        scale *= 2


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2606_00866_b200 import workload as W
    scale = args.scale or _reference_scale(args.config, W, args.f_busy)
    threads = args.ref_threads if args.ref_threads > 0 else 1
    oe = OracleEpochs(args.config, scale, SEED, args.f_busy)
    for _ in range(args.warmup):
        oe.step(threads)
    t_sum, b_sum = 0.0, 0
    for _ in range(args.steps):
        t, b = oe.step(threads)
        t_sum += t; b_sum += b
    v = b_sum / t_sum / 1e9 if t_sum > 0 else 0.0
    sh = oe.cfg.shape
    sample = (f"{args.steps} epochs of {oe.cfg.name} (pools and contexts / {scale}: byte mirrors of "
              f"{oe.cfg.gpu_pool_pages * sh.page_bytes / GIB:.0f} + {oe.cfg.cpu_pool_pages * sh.page_bytes / GIB:.0f} GiB), "
              f"{b_sum / GIB:.1f} GiB migrated host->host, {threads} thread(s)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_sum / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8",
        "data": "synthetic", "config": {"workload": oe.cfg.name, "bj_config": f"configs[{args.config - 1}]", "scale": scale},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                         "host_cores_available": os.cpu_count(), "cpu_model": _cpu_model()},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
def _load_ncu_traffic() -> dict:
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the gather kernel, from the tracked
    summary of the committed ``ncu --set full`` capture (profiles/ncu_traffic.json names the command,
    the launch and its size)."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f)
    except (OSError, ValueError):
        return {}


def _hbm_peak():
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        return float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def link_report(st, link):
    """Achieved fractions of the measured pinned-memcpy peaks over the steps ``st``."""
    ideal = sum(ideal_seconds(s["dem"], s["pro"], link) for s in st)
    meas = sum(s["ms"] for s in st) * 1e-3
    model = sum(memcpy_model_seconds(s["dem"], s["pro"], link) for s in st)
    out = {"frac_of_measured_link_peak": ideal / meas if meas > 0 and ideal > 0 else None,
           "frac_of_pinned_memcpy_model": model / meas if meas > 0 and model > 0 else None}
    if "d2h_streamed" in link and meas > 0:      # the same bound from the streamed (sustained) rates
        sl = dict(link, d2h=link["d2h_streamed"], h2d=link["h2d_streamed"])
        out["frac_of_streamed_link_rate"] = sum(ideal_seconds(s["dem"], s["pro"], sl) for s in st) / meas
    for name, sel in (("demote_only", lambda s: s["dem"] > 0 and s["pro"] == 0),
                      ("promote_only", lambda s: s["pro"] > 0 and s["dem"] == 0),
                      ("bidirectional", lambda s: s["pro"] > 0 and s["dem"] > 0)):
        sub = [s for s in st if sel(s)]
        if sub:
            byt = sum(s["dem"] + s["pro"] for s in sub)
            sec = sum(s["ms"] for s in sub) * 1e-3
            peak = {"demote_only": link["d2h"], "promote_only": link["h2d"]}.get(name)
            ent = {"steps": len(sub), "GBps": byt / sec / 1e9, "GiB": byt / GIB}
            ent["frac"] = (ent["GBps"] / peak) if peak else \
                sum(ideal_seconds(s["dem"], s["pro"], link) for s in sub) / sec
            if not peak:
                ent["frac_of_pinned_memcpy_model"] = \
                    sum(memcpy_model_seconds(s["dem"], s["pro"], link) for s in sub) / sec
            out[name] = ent
    return out


def measure_config(args, cfg, seed, arena, link, steps, warmup, local, barrier, do_e2e=True,
                   gather_reps=20, clocks_on=True, size_matched_leg=True, do_timeline=False):
    """K timed epochs of one config on the CUDA path (device-resident inputs), the same epochs again
    through the public API from host buffers, the in-step roofline of the gather/scatter kernel and
    the standalone device halves.  -> dict of raw totals and derived records."""
    import torch
    from paper_2606_00866_b200 import binding, workload as W
    from paper_2606_00866_b200.harness import GpuRunner
    sh = cfg.shape
    page_b = sh.page_bytes
    hbm_peak, peak_src = _hbm_peak()
    paths = {"auto": 0, "zerocopy": 1, "staged": 2, "copyengine": 3}
    r = GpuRunner(cfg, seed, arena=arena, staging_bytes=args.staging_mib << 20,
                  path_demote=paths[args.path_demote], path_promote=paths[args.path_promote],
                  copy_kernel={"auto": 0, "ldst": 1, "tma": 2}[args.kernel])
    sim = W.Sim(cfg, seed)
    cur = torch.cuda.current_stream()
    sticky = args.policy == "sticky"

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def epoch(mode):
        """One step.  mode 'dev': inputs resident, regions A+B timed; 'e2e': host buffers, one
        region.  -> dict(ms, dem, pro, h2d, d2h)."""
        plan = sim.begin_epoch()                                   # input generation (host)
        n = cfg.n_programs
        if mode == "dev":
            r.upload_inputs(plan.iota, plan.kv_pages, plan.prev_tier)
            torch.cuda.synchronize()
            a0, a1, b0, b1 = ev(), ev(), ev(), ev()
            a0.record(cur)
            if sticky:                                             # NEXT-1 policy: status flags ride along
                got = r.place_sticky(plan.iota, plan.kv_pages, plan.prev_tier, plan.flags, stream=cur)
            else:
                got = r.place_resident(cur, done_event=a1)         # kernel (+ D2H of the lists), then sync
            if sticky:
                a1.record(cur)
            sim.apply_placement(got["tier"], got["lists"])         # harness allocator (untimed) ...
            prepared = r.prepare(plan)                             # ... and the calls' page / slot tables
            if timeline is not None:
                r.mori.mori_profile(2)                             # time zero of this step's timeline
            b0.record(cur)
            r.mori.mori_after_stream(binding.BOTH, cur)
            r.issue(prepared, sync=False)
            r.mori.mori_stream_wait(cur, binding.BOTH)
            b1.record(cur)
            r.mori.mori_sync(binding.BOTH)
            torch.cuda.synchronize()
            ms_a, ms_b = a0.elapsed_time(a1), b0.elapsed_time(b1)
            ms = ms_a + ms_b
            if timeline is not None:
                timeline.append({"demote_bytes": plan.demote_pages * page_b, "promote_bytes": plan.promote_pages * page_b,
                                 "region_b_ms": b0.elapsed_time(b1),
                                 "rows": "kind 0 = gather/scatter kernel, 1 = one staging segment's DMAs; [kind, start_ms, end_ms, bytes]",
                                 "demote": r.mori.mori_profile_timeline(binding.DEMOTE),
                                 "promote": r.mori.mori_profile_timeline(binding.PROMOTE)})
        else:
            torch.cuda.synchronize()
            e0, e1 = ev(), ev()
            e0.record(cur)
            r.mori.mori_after_stream(binding.BOTH, cur)
            got = (r.place_sticky(plan.iota, plan.kv_pages, plan.prev_tier, plan.flags, stream=cur) if sticky
                   else r.place(plan.iota, plan.kv_pages, plan.prev_tier, stream=cur))
            sim.apply_placement(got["tier"], got["lists"])
            r.execute(plan, sync=False)
            r.mori.mori_stream_wait(cur, binding.BOTH)
            e1.record(cur)
            r.mori.mori_sync(binding.BOTH)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
        sim.end_epoch()
        r.fill(plan.fills)                                          # stands in for prefill (untimed)
        n_tab = 8 * (plan.demote_pages + plan.promote_pages)        # page + slot ids, int32 each
        return dict(ms=ms, ms_b=ms_b if mode == "dev" else None, ops=[(op[0][0], len(op[3])) for op in plan.ops if op[0] != "sync_all"],
                    dem=plan.demote_pages * page_b, pro=plan.promote_pages * page_b,
                    h2d=plan.promote_pages * page_b + 9 * n + n_tab,
                    d2h=plan.demote_pages * page_b + r.h_out.numel())

    timeline = None
    for _ in range(warmup):
        epoch("dev")
    timeline = [] if (do_timeline and getattr(args, "timeline", None)) else None
    # ---- timed: K steps, device-resident inputs ---------------------------------------------------
    r.mori.mori_profile(True)
    r.mori.mori_profile_read(binding.DEMOTE); r.mori.mori_profile_read(binding.PROMOTE)
    clocks = ClockSampler(local) if clocks_on else None
    barrier()
    if clocks:
        clocks.start()
    l0 = r.mori.mori_launch_count()
    st = [epoch("dev") for _ in range(steps)]
    barrier()
    launches = r.mori.mori_launch_count() - l0
    clk = clocks.stop() if clocks else None
    prof = {"demote": r.mori.mori_profile_read(binding.DEMOTE),
            "promote": r.mori.mori_profile_read(binding.PROMOTE)}
    r.mori.mori_profile(False)
    if timeline is not None:
        with open(args.timeline, "w") as f:
            json.dump({"workload": cfg.name, "how": "bench.py --timeline: CUDA events the library records around every "
                       "kernel and every staging segment's DMAs, milliseconds since the start of the step's region B",
                       "link_peaks_GBps": link, "steps": timeline}, f)
        timeline = None
    if args.verbose:
        for i, x in enumerate(st):
            gb = (x["dem"] + x["pro"]) / 1e9
            print(f"{cfg.name} step {i}: {x['ms']:.3f} ms  demote {x['dem'] / GIB:.2f} GiB  promote {x['pro'] / GIB:.2f} GiB  "
                  f"{gb / (x['ms'] * 1e-3) if x['ms'] > 0 else 0:.1f} GB/s  ops {x['ops']}", file=sys.stderr)
    # ---- timed: the SAME epochs again through the public API from host buffers (the trace and the
    #      placement are deterministic in the seed, so `e2e` and `value` move identical bytes) -------
    st_e2e = []
    if do_e2e:
        sim = W.Sim(cfg, seed)
        for _ in range(warmup):
            epoch("e2e")
        barrier()
        st_e2e = [epoch("e2e") for _ in range(steps)]
        barrier()

    def total(x, k):
        return float(sum(s_[k] for s_ in x))

    out = {"cfg": cfg, "runner_paths": r.mori_paths, "kernel_name": binding.KERNEL_NAMES[r.mori.copy_kernel],
           "steps": st, "steps_e2e": st_e2e, "launches": launches, "clocks": clk,
           "t_dev": total(st, "ms") * 1e-3, "b_dev": total(st, "dem") + total(st, "pro"),
           "t_e2e": total(st_e2e, "ms") * 1e-3, "b_e2e": total(st_e2e, "dem") + total(st_e2e, "pro"),
           "h2d_per_step": total(st_e2e, "h2d") / max(1, len(st_e2e)),
           "d2h_per_step": total(st_e2e, "d2h") / max(1, len(st_e2e))}

    # ---- size-matched peak: a plain pinned memcpy of ONE epoch's mean bytes; for GiB-
    #      sized epochs it equals the asymptotic peak, for cfg 1's KiB-sized ones it is what
    #      "latency-bound" means on this link ---------------------------------------------------------
    moving = [x for x in st if x["dem"] + x["pro"] > 0]
    out["moving_steps"] = len(moving)
    out["size_matched"] = None
    if moving and size_matched_leg:
        mean_b = int(sum(x["dem"] + x["pro"] for x in moving) / len(moving))
        mean_b = max(4096, min(mean_b, arena.numel() // 2, 2 * GIB)) // 4096 * 4096
        sm = measure_link_peak(arena, nbytes=mean_b, reps=10)
        ach = sum(x["dem"] + x["pro"] for x in moving) / (sum(x["ms"] for x in moving) * 1e-3) / 1e9
        ach_b = sum(x["dem"] + x["pro"] for x in moving) / (sum(x["ms_b"] for x in moving) * 1e-3) / 1e9
        smj = measure_link_peak(arena, nbytes=mean_b, reps=10, joined=True) if mean_b < (64 << 20) else sm
        out["size_matched"] = {"bytes": mean_b, "d2h_GBps": sm["d2h"], "h2d_GBps": sm["h2d"],
                               "d2h_joined_GBps": smj["d2h"], "transfer_region_over_d2h_joined": ach_b / smj["d2h"],
                               "epochs_GBps": ach, "epochs_over_d2h": ach / sm["d2h"],
                               "transfer_region_GBps": ach_b, "transfer_region_over_d2h": ach_b / sm["d2h"],
                               "note": "one-direction denominator: epochs that move both ways can exceed it; "
                                       "`epochs` = rank/partition + transfers, `transfer_region` = the demote/promote "
                                       "calls up to the join only (what a plain memcpy of the same bytes competes with); "
                                       "`joined` = the same memcpy issued on a side stream and joined to the timing stream "
                                       "on both ends, as an epoch's transfers are"}

    # ---- roofline of the HBM-bound kernel, from the library's per-launch CUDA events ---------------
    ncu = _load_ncu_traffic()
    k_ms = prof["demote"][0] + prof["promote"][0]
    k_n = prof["demote"][1] + prof["promote"][1]
    k_b = prof["demote"][2] + prof["promote"][2]
    staged_bytes = sum(x["dem"] + x["pro"] for x in st)
    roofline = None
    if binding.PATH_STAGED in r.mori_paths and k_ms > 0 and k_b >= 0.5 * staged_bytes and k_b / k_n > (64 << 20):
        ach = 2.0 * k_b / (k_ms * 1e-3) / 1e9                     # read + write, per DESIGN.md 5
        roofline = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                    "traffic": ncu.get("dram_bytes_per_launch"),
                    "kernel": f"copy_pages_{binding.KERNEL_NAMES[r.mori.copy_kernel]}"
                              " (gather/scatter of the STAGED path, inside the timed steps)",
                    "peak_source": peak_src, "traffic_source": ncu.get("source"),
                    "traffic_launch_algorithmic_bytes": ncu.get("algorithmic_bytes_same_launch"),
                    "traffic_over_algorithmic_same_launch": ncu.get("ratio"),
                    "launches": k_n, "avg_launch_us": 1e3 * k_ms / k_n,
                    "algorithmic_bytes_per_launch": 2.0 * k_b / k_n}
    out["roofline"] = roofline
    # ---- the device halves alone: pool <-> contiguous device buffer, >= 4 GiB per launch ------------
    out["gather_scatter"] = gather_scatter_leg(r, sim, hbm_peak, reps=gather_reps) if gather_reps > 0 else None
    out["free_gpu_pages"] = max(0, cfg.cap_gpu_pages - int(sum(p_.size for p_ in sim.gpu_pages)))
    out["runner"] = r
    return out


def _per_config_record(m, link, scale):
    """The compact per-config sub-record of the bench line (north_star: "reported per config as an
    absolute number and as a fraction of the measured pinned-memcpy host-link peak")."""
    cfg = m["cfg"]
    sh = cfg.shape
    lr = link_report(m["steps"], link)
    rec = {"workload": cfg.name, "bj_config": f"configs[{cfg.index - 1}]", "scale": scale, "f_busy": cfg.f_busy,
           "GBps": m["b_dev"] / m["t_dev"] / 1e9 if m["t_dev"] > 0 else 0.0,
           "frac_of_measured_link_peak": lr["frac_of_measured_link_peak"],
           "frac_of_pinned_memcpy_model": lr["frac_of_pinned_memcpy_model"],
           "e2e_GBps": m["b_e2e"] / m["t_e2e"] / 1e9 if m["t_e2e"] > 0 else None,
           "steps": len(m["steps"]), "moving_steps": m["moving_steps"], "migrated_GiB": m["b_dev"] / GIB,
           "ms_per_step": 1e3 * m["t_dev"] / max(1, len(m["steps"])),
           "ranker_capacity_pages": {"gpu": cfg.cap_gpu_pages, "cpu": cfg.cap_cpu_pages,
                                     "gpu_GiB": cfg.cap_gpu_pages * sh.page_bytes / GIB,
                                     "note": "physical pool minus headroom (DESIGN.md R23)"},
           "pools_GiB": {"gpu": cfg.gpu_pool_pages * sh.page_bytes / GIB, "cpu": cfg.cpu_pool_pages * sh.page_bytes / GIB},
           "paths": [PATH_NAME.get(x, str(x)) for x in m["runner_paths"]], "gpu_launches": int(m["launches"])}
    for k in ("demote_only", "promote_only", "bidirectional"):
        if k in lr:
            rec[k] = {"steps": lr[k]["steps"], "GBps": lr[k]["GBps"], "frac": lr[k]["frac"]}
    if m["size_matched"]:
        smx = m["size_matched"]
        rec["size_matched"] = {"bytes": smx["bytes"], "pinned_memcpy_GBps": smx["d2h_GBps"],
                               "epochs_GBps": smx["epochs_GBps"], "frac": smx["epochs_over_d2h"],
                               "transfer_region_GBps": smx["transfer_region_GBps"],
                               "transfer_region_frac": smx["transfer_region_over_d2h"],
                               "pinned_memcpy_joined_GBps": smx["d2h_joined_GBps"],
                               "transfer_region_frac_of_joined_memcpy": smx["transfer_region_over_d2h_joined"]}
    if m["roofline"]:
        rec["in_step_gather_scatter_frac_of_measured_hbm"] = m["roofline"]["frac"]
        rec["in_step_launches"] = m["roofline"]["launches"]
    gs = m["gather_scatter"]
    if gs:
        rec["standalone_gather_frac_of_measured_hbm"] = gs["gather_frac_of_measured_hbm"]
        rec["standalone_scatter_frac_of_measured_hbm"] = gs["scatter_frac_of_measured_hbm"]
        rec["standalone_GiB_per_launch"] = gs["GiB_per_launch"]
    return rec


PATH_NAME = {1: "zerocopy", 2: "staged", 3: "copyengine"}


def _fit_scale(cfg_index: int, world: int, W, f_busy=None) -> int:
    """SURVEY 8(d) scale rule: the smallest power of two that lets the pinned arena fit host RAM and
    the pool fit HBM.  One replica: the arena plus 20 GiB must fit MemAvailable (cfg 3's 160 GiB does
    on a 196 GiB box, cfg 4's 200 GiB does not).  Several replicas share the node: 70 % of MemTotal
    divided by the ranks (MemTotal so that every rank picks the same scale)."""
    import torch
    if world > 1:
        avail = int(_meminfo_kb("MemTotal") * 1024 * 0.70) // world
    else:
        avail = _meminfo_kb("MemAvailable") * 1024 - 20 * GIB
    free_hbm, _ = torch.cuda.mem_get_info()
    scale = 1
    while True:
        cfg = W.get_config(cfg_index, scale, f_busy)
        sh = cfg.shape
        if (cfg.cpu_pool_pages * sh.page_bytes <= avail
                and cfg.gpu_pool_pages * sh.page_bytes + (5 << 30) <= free_hbm):
            return scale
        scale *= 2


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_00866_b200 import binding, replicas, workload as W

    rank, world, local = replicas.env_rank()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    if args.device_index >= 0:
        local = args.device_index                    # testing only: several replicas on one GPU
    torch.cuda.set_device(local)
    if world > 1:
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(args.backend)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- which configs run: the headline one (BASELINE.json configs[1] unless --config), then, on a
    #      default single-GPU run, every other config of BASELINE.json as a `per_config` sub-record ----
    scale = args.scale or _fit_scale(args.config, world, W, args.f_busy)
    cfg = W.get_config(args.config, scale, args.f_busy)
    others = []
    if args.per_config and world == 1 and rank == 0:
        for idx, fb in ((1, None), (3, 0.25), (3, 0.5), (3, 0.75), (4, None), (5, None), (2, None)):
            if idx == args.config and (fb == args.f_busy or idx != 3):
                continue
            others.append((idx, fb, 1 if idx == 1 else _fit_scale(idx, world, W, fb)))
    sh = cfg.shape
    seed = replicas.replica_seed(SEED, rank)
    t_setup = time.perf_counter()
    thp0 = _meminfo_kb("AnonHugePages")
    def _arena_bytes(i, sc, fb):
        c_ = W.get_config(i, sc, fb)
        return c_.cpu_pool_pages * c_.shape.page_bytes

    own_bytes = cfg.cpu_pool_pages * sh.page_bytes
    arena_bytes = max([own_bytes] + [_arena_bytes(i, sc, fb) for i, fb, sc in others])
    try:
        arena_full = binding.Mori.mori_host_alloc(arena_bytes)      # ONE pinned arena serves every config
    except binding.MoriError as e:
        # the box refuses to page-lock the largest arena (cfg 3's 160 GiB): the side legs that need more than
        # the headline's arena drop to the smallest scale that fits it, and say so in their records
        print(f"NOTE pinning {arena_bytes / GIB:.0f} GiB refused ({e}); per_config legs limited to "
              f"{own_bytes / GIB:.0f} GiB arenas", file=sys.stderr)
        shrunk = []
        for i, fb, sc in others:
            while _arena_bytes(i, sc, fb) > own_bytes:
                sc *= 2
            shrunk.append((i, fb, sc))
        others = shrunk
        arena_full = binding.Mori.mori_host_alloc(own_bytes)
    arena_thp_gib = (_meminfo_kb("AnonHugePages") - thp0) / (1 << 20)
    link = measure_link_peak(arena_full, stream_chunks=16)
    t_setup = time.perf_counter() - t_setup
    hbm_peak, peak_src = _hbm_peak()
    page_b = sh.page_bytes

    m = measure_config(args, cfg, seed, arena_full[:cfg.cpu_pool_pages * page_b], link, args.steps, args.warmup,
                       local, barrier, do_e2e=True, gather_reps=0 if (args.no_gather_leg or rank != 0) else 20,
                       do_timeline=(rank == 0))
    r = m["runner"]
    (t_dev, t_e2e), (b_dev, b_e2e, launches) = replicas.aggregate(
        [m["t_dev"], m["t_e2e"]], [m["b_dev"], m["b_e2e"], float(m["launches"])], device="cuda")
    value = b_dev / t_dev / 1e9 if t_dev > 0 else 0.0
    value_e2e = b_e2e / t_e2e / 1e9 if t_e2e > 0 else 0.0
    roofline, gs = m["roofline"], m["gather_scatter"]
    if roofline is None and gs:
        ncu = _load_ncu_traffic()
        roofline = {"bound": "hbm", "achieved": gs["gather_GBps"], "peak": hbm_peak, "unit": "GB/s",
                    "frac": gs["gather_GBps"] / hbm_peak, "traffic": ncu.get("dram_bytes_per_launch"),
                    "kernel": gs["kernel"] + " (standalone gather launches)", "peak_source": peak_src,
                    "traffic_source": ncu.get("source")}

    # ---- the shared Waiting queue across replicas: all-gather every replica's
    #      free GPU pages (NCCL; stays on the device) and pack the same queue on every rank ---------
    free_all = replicas.gather_free_capacity(m["free_gpu_pages"], device="cuda")
    wq_rng = np.random.default_rng(SEED)                             # one queue, identical on every rank
    wq_n = cfg.n_programs                                            # (the context is sized for n programs)
    wq = [torch.from_numpy(x).cuda() for x in (
        wq_rng.integers(1, max(2, cfg.max_program_pages // 4), wq_n).astype(np.int32),
        wq_rng.random(wq_n).astype(np.float32), (2 | (wq_rng.integers(0, 2, wq_n) * 4)).astype(np.uint8))]
    wq_rep = torch.empty(wq_n, dtype=torch.int32, device="cuda")
    wq_left = torch.empty_like(free_all)
    r.mori.mori_bfd_assign(wq[0], wq[1], wq[2], free_all, wq_rep, wq_left)
    torch.cuda.synchronize()
    waiting_queue = {"replicas": int(free_all.numel()), "free_pages": free_all.tolist(), "candidates": wq_n,
                     "admitted_here": int((wq_rep == rank).sum().item()),
                     "admitted_total": int((wq_rep >= 0).sum().item()), "free_pages_left": wq_left.tolist()}
    r.close()
    m["runner"] = None
    del r
    torch.cuda.empty_cache()

    # ---- every other BASELINE.json config, driver-timed in the same run (single GPU only) ----------
    per_config = [_per_config_record(m, link, scale)]
    for idx, fb, sc in others:
        t0 = time.perf_counter()
        try:
            c2 = W.get_config(idx, sc, fb)
            # the box is one GPU of a shared host and its pinned-memcpy rate drifts within a run: every leg
            # is held against peaks measured right before it (both sets are printed)
            link2 = measure_link_peak(arena_full, reps=3)
            m2 = measure_config(args, c2, seed, arena_full[:c2.cpu_pool_pages * c2.shape.page_bytes], link2,
                                args.per_config_steps if idx != 1 else c2.epochs - 4, 4, local, barrier,
                                do_e2e=(idx == 1), gather_reps=0 if (args.no_gather_leg or idx == 1) else 5,
                                clocks_on=False)
            m2["runner"].close()
            m2["runner"] = None
            rec = _per_config_record(m2, link2, sc)
            rec["link_peaks_GBps_before_leg"] = {k: link2[k] for k in ("d2h", "h2d", "bidir_sum")}
            rec["frac_of_link_peak_measured_at_start"] = link_report(m2["steps"], link)["frac_of_measured_link_peak"]
            rec["leg_seconds"] = time.perf_counter() - t0
            per_config.append(rec)
            del m2
        except Exception as e:                                       # a failed side leg must not lose the headline
            per_config.append({"workload": f"cfg{idx}" + (f"-f{fb:g}" if fb else ""), "scale": sc,
                               "error": f"{type(e).__name__}: {e}"})
        torch.cuda.empty_cache()
    per_config.sort(key=lambda x: x.get("workload", ""))
    binding.Mori.mori_host_free(arena_full)

    with_oracle = world == 1 and not args.no_cpu_baseline
    rp = rank_partition_leg(with_oracle=with_oracle) if rank == 0 else None
    evl = eviction_leg(with_oracle=with_oracle) if rank == 0 else None
    sml = small_move_leg() if rank == 0 else None
    cpu = None
    if rank == 0 and with_oracle:
        cpu = cpu_baseline(args.config, f_busy=args.f_busy)
        if args.per_config:
            cpu["per_config"] = []
            for idx, fb, sc in others:
                try:
                    cb = cpu_baseline(idx, budget_s=2.0, f_busy=fb, max_bytes=6 * GIB)
                    cpu["per_config"].append({"workload": cb["workload"], "scale": cb["scale"], "GBps_1_core": cb["value"],
                                              "GBps_all_cores": cb["all_cores"]["value"], "cores": cb["all_cores"]["cores"]})
                except Exception as e:
                    cpu["per_config"].append({"workload": f"cfg{idx}", "error": f"{type(e).__name__}: {e}"})
    if rank == 0:
        K = args.steps
        lr = link_report(m["steps"], link)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT,
            "frac_of_measured_link_peak": lr["frac_of_measured_link_peak"],
            "roofline_frac": roofline["frac"] if roofline else None,
            "n_gpus": world, "steps": K,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_dev / K, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": cfg.name, "bj_config": f"configs[{args.config - 1}]", "scale": scale,
                       "n_programs": cfg.n_programs, "gpu_pool_GiB": cfg.gpu_pool_pages * page_b / GIB,
                       "host_arena_GiB": cfg.cpu_pool_pages * page_b / GIB,
                       "ranker_gpu_capacity_GiB": cfg.cap_gpu_pages * page_b / GIB,
                       "ranker_cpu_capacity_GiB": cfg.cap_cpu_pages * page_b / GIB,
                       "page_bytes": page_b, "chunk_bytes": sh.chunk_bytes,
                       "parallelism": f"replicas x{world} (no data-path collective)",
                       "path_demote": binding.PATH_NAMES[m["runner_paths"][0]],
                       "path_promote": binding.PATH_NAMES[m["runner_paths"][1]],
                       "copy_kernel": m["kernel_name"],
                       "staging_MiB": args.staging_mib, "policy": args.policy,
                       "l2": "inputs larger than L2 (GiB per step vs 126 MB); no flush needed",
                       "migrated_GiB": b_dev / GIB, "setup_s": t_setup,
                       "host_arena_on_huge_pages_GiB": arena_thp_gib},
            "clocks": m["clocks"],
            "e2e": {"value": value_e2e, "unit": UNIT,
                    "h2d_bytes_per_step": m["h2d_per_step"],
                    "d2h_bytes_per_step": m["d2h_per_step"],
                    "ms_per_step": 1e3 * t_e2e / K, "migrated_GiB": b_e2e / GIB,
                    "link": link_report(m["steps_e2e"], link)},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "per_config": per_config,
            "link": dict(lr, peaks_GBps=link, size_matched=m["size_matched"],
                         peak_how="pinned cudaMemcpyAsync of one contiguous 1 GiB buffer, best of 5, "
                                  "measured in this process before the run"),
            "gather_scatter": gs,
            "rank_partition": rp,
            "eviction_order": evl,
            "small_move": sml,
            "waiting_queue_bfd": waiting_queue,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    if world > 1:
        dist.barrier()                      # rank 0 is still running its single-rank legs
        dist.destroy_process_group()


def gather_scatter_leg(r, sim, hbm_peak, min_bytes=4 * GIB, reps=20, warm=3):
    """mori_gather_pages / mori_scatter_pages on the page tables the workload has produced
    (resident GPU-tier programs, in table order), padded with the remaining pool pages in
    allocator order up to >= 4 GiB: one launch, CUDA events on the launching stream."""
    import torch
    from paper_2606_00866_b200 import binding
    cfg, sh = r.cfg, r.cfg.shape
    pages = [p for p in sim.gpu_pages if p.size]
    used = np.concatenate(pages) if pages else np.zeros(0, np.int32)
    want = -(-min_bytes // sh.page_bytes)
    if used.size < want:
        rest = np.setdiff1d(np.arange(cfg.gpu_pool_pages, dtype=np.int32), used)
        used = np.concatenate([used, rest[:want - used.size]])
    used = used[:max(want, 1)].astype(np.int32)
    free, _ = torch.cuda.mem_get_info()
    n = int(min(used.size, (free - GIB) // sh.page_bytes))
    if n <= 0:
        return None
    used = used[:n]
    gd = torch.from_numpy(used).cuda()
    buf = torch.empty(n * sh.page_bytes, dtype=torch.uint8, device="cuda")
    cur = torch.cuda.current_stream()
    out = {"pages": n, "GiB_per_launch": n * sh.page_bytes / GIB,
           "kernel": f"copy_pages_{binding.KERNEL_NAMES[r.mori.copy_kernel]}",
           "contiguous_runs_mean_pages": float(n / max(1, 1 + np.count_nonzero(np.diff(used) != 1)))}
    for name, fn in (("gather", lambda: r.mori.mori_gather_pages(gd, buf, stream=cur)),
                     ("scatter", lambda: r.mori.mori_scatter_pages(gd, buf, stream=cur))):
        for _ in range(warm):
            fn()
        ts = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(cur); fn(); e1.record(cur)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        byt = 2.0 * n * sh.page_bytes
        out[f"{name}_GBps"] = byt / float(np.median(ts)) / 1e9
        out[f"{name}_GBps_best"] = byt / min(ts) / 1e9
        out[f"{name}_frac_of_measured_hbm"] = out[f"{name}_GBps"] / hbm_peak
        out[f"{name}_frac_of_8TBps_spec"] = out[f"{name}_GBps"] / 8000.0
    del buf
    return out


def copy_kernel_sweep(args):
    """`--leg copy_sweep`: the gather/scatter kernel ALONE (1 / 2 / 4 GiB per launch) and IN-STEP (inside
    a STAGED demotion, a STAGED promotion and both at once, i.e. next to the copy engines' DMA), for
    the ring geometries, chunk hand-out and staging sizes that DESIGN.md section 7 discusses.  cfg-2
    geometry on a 28 GiB pool and a 16 GiB pinned arena.  One JSON line: rows of fractions of the
    measured HBM copy rate."""
    import itertools
    import torch
    from paper_2606_00866_b200 import binding
    L, H, D, T = 32, 8, 128, 16
    page = L * 2 * H * T * D * 2
    P, S = 14336, 8192
    pool = torch.empty(P * page, dtype=torch.uint8, device="cuda")
    pool.random_(0, 255)
    arena = binding.Mori.mori_host_alloc(S * page)
    peak, peak_src = _hbm_peak()
    rng = np.random.default_rng(0)
    cur = torch.cuda.current_stream()
    variants = [(sched, piece, ctas, stg, "tma")
                for sched, piece, ctas, stg in itertools.product((1, 0), (64, 32, 16), (1, 2), (1024, 2048))
                if not (ctas == 2 and piece == 64) and not (sched == 0 and (ctas == 2 or piece != 64))]
    variants += [(1, 64, 1, 1024, "ldst"), (1, 64, 1, 2048, "ldst")]
    rows = []
    for sched, piece, ctas, stg, kern in variants:
        os.environ.update(MORI_SCHED=str(sched), MORI_PIECE_KIB=str(piece), MORI_CTAS_PER_SM=str(ctas))
        m = binding.Mori(L, H, D, T, pool, arena, path_demote=2, path_promote=2,
                         copy_kernel={"tma": 2, "ldst": 1}[kern], staging_bytes=stg << 20)
        row = dict(kernel=kern, chunk_handout="dynamic" if sched else "static", piece_KiB=piece, ctas_per_sm=ctas,
                   staging_MiB=stg)
        for gib in (1, 2, 4):
            n = gib * GIB // page
            g = torch.from_numpy(rng.permutation(P)[:n].astype(np.int32)).cuda()
            buf = torch.empty(n * page, dtype=torch.uint8, device="cuda")
            ts = []
            for _ in range(8):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(cur); m.mori_gather_pages(g, buf, stream=cur); e1.record(cur); torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            row[f"alone_{gib}GiB_us"] = 1e3 * float(np.median(ts[2:]))
            row[f"alone_{gib}GiB_frac"] = 2 * n * page / (np.median(ts[2:]) * 1e-3) / 1e9 / peak
            del buf
        n = 6144                                                     # 12 GiB
        for mode in ("demote", "promote", "both"):
            g = rng.permutation(P)[:n].astype(np.int32)
            g2 = np.setdiff1d(np.arange(P, dtype=np.int32), g)[:n]
            h = np.arange(n, dtype=np.int32)
            m.mori_profile(True); m.mori_profile_read(1); m.mori_profile_read(2)
            if mode == "demote":
                m.mori_demote(g, h)
            elif mode == "promote":
                m.mori_promote(h, g2)
            else:
                m.mori_demote(g[:n // 2], h[:n // 2]); m.mori_promote(h[n // 2:], g2[:n - n // 2])
            m.mori_sync(3)
            pd, pp = m.mori_profile_read(1), m.mori_profile_read(2)
            ms, nl, nb = pd[0] + pp[0], pd[1] + pp[1], pd[2] + pp[2]
            row[f"instep_{mode}_frac"] = 2 * nb / (ms * 1e-3) / 1e9 / peak
            row[f"instep_{mode}_us_per_launch"] = 1e3 * ms / nl
        m.close()
        rows.append(row)
    for k in ("MORI_SCHED", "MORI_PIECE_KIB", "MORI_CTAS_PER_SM"):
        os.environ.pop(k, None)
    binding.Mori.mori_host_free(arena)
    print(json.dumps({"leg": "copy_sweep", "hbm_peak_GBps": peak, "peak_source": peak_src,
                      "geometry": "cfg 2 (32 layers, 64 KiB chunks, 2 MiB pages), 28 GiB pool, 16 GiB pinned arena, "
                                  "random page ids, consecutive slots", "rows": rows}))


def three_tier_leg(args):
    """`--leg three_tier`: the movers of a three-tier hierarchy (GPU pool, a middle arena in device memory
    -- a second buffer of this GPU standing in for a peer GPU's HBM -- and the pinned host arena;
    P:L339-351) one pair and one direction at a time, 4 GiB per move, then whole epochs driven by
    mori_rank_partition_tiers.  cfg 2 at scale 4.  One JSON line."""
    import torch
    from paper_2606_00866_b200 import binding, workload as W
    from paper_2606_00866_b200.harness import TierRunner
    cfg = W.get_config(2, args.scale or 4)
    sh = cfg.shape
    mid_ids = cfg.gpu_pool_pages // 2
    arena = binding.Mori.mori_host_alloc(cfg.cpu_pool_pages * sh.page_bytes)
    r = TierRunner(cfg, SEED, mid_ids, host_arena=arena)
    r.pool.random_(0, 255)
    rng = np.random.default_rng(SEED)
    n = int(min(4 * GIB // sh.page_bytes, mid_ids, cfg.gpu_pool_pages // 2, cfg.cpu_pool_pages // 2))
    cur = torch.cuda.current_stream()
    pairs = {}
    for name, ctx, n_fast, n_slow in (("pool_mid", r.pool_mid, cfg.gpu_pool_pages, mid_ids),
                                      ("pool_host", r.pool_host, cfg.gpu_pool_pages, cfg.cpu_pool_pages),
                                      ("mid_host", r.mid_host, mid_ids, cfg.cpu_pool_pages)):
        fast = rng.permutation(n_fast)[:n].astype(np.int32)          # scattered ids in the faster pool
        slow = np.arange(n, dtype=np.int32)                          # one run of slots in the slower one
        ent = {}
        for direction in ("down", "up"):
            ts = []
            for _ in range(4):
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(cur)
                ctx.mori_after_stream(binding.BOTH, cur)
                if direction == "down":
                    ctx.mori_demote(fast, slow, want_ticket=False)
                else:
                    ctx.mori_promote(slow, fast, want_ticket=False)
                ctx.mori_stream_wait(cur, binding.BOTH)
                e1.record(cur)
                ctx.mori_sync(binding.BOTH)
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e-3)
            ent[direction + "_GBps"] = n * sh.page_bytes / float(np.median(ts[1:])) / 1e9
        ent["GiB_per_move"] = n * sh.page_bytes / GIB
        pairs[name] = ent
    # whole epochs: placement by mori_rank_partition_tiers, bytes by the three pair-contexts
    r.pool.zero_()
    pool_ids = [cfg.gpu_pool_pages, mid_ids, cfg.cpu_pool_pages]
    caps = [cfg.cap_gpu_pages, mid_ids - cfg.max_program_pages // 2, cfg.cap_cpu_pages]
    sim = W.SimTiers(cfg, SEED, pool_ids, caps)
    moved = {}
    t_move, epochs = 0.0, 0
    for e in range(args.warmup + args.steps):
        plan = sim.begin_epoch()
        got = r.place(plan.iota, plan.kv_pages, plan.prev_tier, caps)
        sim.apply_placement(got["tier"], got["moves"])
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r.execute(plan)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        sim.end_epoch()
        r.fill(plan.fills)
        if e >= args.warmup:
            t_move += dt; epochs += 1
            for op in plan.ops:
                if op[0] == "move":
                    k = f"{op[2]}->{op[3]}"
                    moved[k] = moved.get(k, 0) + len(op[4]) * sh.page_bytes
    tot = sum(moved.values())
    r.close()
    binding.Mori.mori_host_free(arena)
    print(json.dumps({"leg": "three_tier", "workload": cfg.name, "tiers": "0 = GPU pool, 1 = middle arena (device memory of the "
                      "SAME GPU: stands in for peer HBM; NVLink bandwidth unmeasured, one GPU), 2 = pinned host arena",
                      "pools_GiB": [x * sh.page_bytes / GIB for x in pool_ids], "pairs": pairs,
                      "epochs": {"timed": epochs, "moved_GiB_by_pair": {k: v / GIB for k, v in sorted(moved.items())},
                                 "GBps_all_pairs_host_timed": tot / t_move / 1e9 if t_move > 0 else 0.0,
                                 "note": "host wall-clock around TierRunner.execute (three contexts, joins included)"}}))


def small_move_leg(reps=60):
    """The one-launch path of a small move, warm: cfg 1's geometry (16 KiB pages) and the 17-page
    (272 KiB) demotion its trace produces, repeated through the C ABI with the same bracketing an
    epoch's transfer region has (event, mori_after_stream, mori_demote / mori_promote,
    mori_stream_wait, event) -- median device microseconds -- beside a plain pinned memcpy of the
    same bytes, alone between two events and joined through a side stream the same way.  cfg 1's own
    epochs contain this move exactly once, cold (no move in its warm-up epochs)."""
    import torch
    from paper_2606_00866_b200 import binding
    L, H, D, T, P, S = 2, 2, 64, 16, 64, 256
    page = L * 2 * H * T * D * 2
    pool = torch.zeros(P * page, dtype=torch.uint8, device="cuda")
    arena = torch.zeros(S * page, dtype=torch.uint8).pin_memory()
    m = binding.Mori(L, H, D, T, pool, arena)
    cur = torch.cuda.current_stream()
    rng = np.random.default_rng(SEED)
    n = 17
    g = np.ascontiguousarray(rng.permutation(P)[:n], dtype=np.int32)
    h = np.arange(n, dtype=np.int32)
    lib, hc = m._lib, m._h

    def region(fn):
        ts = []
        for _ in range(reps):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(cur)
            m.mori_after_stream(binding.BOTH, cur)
            fn()
            m.mori_stream_wait(cur, binding.BOTH)
            e1.record(cur)
            m.mori_sync(binding.BOTH)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        return float(np.median(ts[5:]))
    dem_us = region(lambda: lib.mori_demote(hc, n, g.ctypes.data, h.ctypes.data, 0, None))
    pro_us = region(lambda: lib.mori_promote(hc, n, h.ctypes.data, g.ctypes.data, 0, 0, None))
    nbytes = n * page
    d_buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    h_buf = arena[:nbytes]
    side = torch.cuda.Stream()

    def memcpy(joined, d2h):
        ts = []
        for _ in range(reps):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(cur)
            if joined:
                side.wait_event(e0)
                with torch.cuda.stream(side):
                    (h_buf.copy_(d_buf, non_blocking=True) if d2h else d_buf.copy_(h_buf, non_blocking=True))
                cur.wait_stream(side)
            else:
                (h_buf.copy_(d_buf, non_blocking=True) if d2h else d_buf.copy_(h_buf, non_blocking=True))
            e1.record(cur)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        return float(np.median(ts[5:]))
    out = {"pages": n, "bytes": nbytes, "demote_us": dem_us, "promote_us": pro_us,
           "memcpy_d2h_bare_us": memcpy(False, True), "memcpy_d2h_joined_us": memcpy(True, True),
           "memcpy_h2d_bare_us": memcpy(False, False), "memcpy_h2d_joined_us": memcpy(True, False)}
    out["demote_GBps"] = nbytes / dem_us / 1e3
    out["promote_GBps"] = nbytes / pro_us / 1e3
    out["demote_frac_of_joined_memcpy"] = out["memcpy_d2h_joined_us"] / dem_us
    out["promote_frac_of_joined_memcpy"] = out["memcpy_h2d_joined_us"] / pro_us
    out["demote_frac_of_bare_memcpy"] = out["memcpy_d2h_bare_us"] / dem_us
    out["promote_frac_of_bare_memcpy"] = out["memcpy_h2d_bare_us"] / pro_us
    m.close()
    return out


def launch_floor(m, cur, reps=200):
    """The floor the latency-bound entry points are judged against: an EMPTY kernel (mori_noop)
    launched through the same binding on the same stream -- device microseconds per call over `reps`
    back-to-back launches, and host wall-clock of one launch + stream synchronize."""
    import torch
    for _ in range(10):
        m.mori_noop(stream=cur)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(cur)
    for _ in range(reps):
        m.mori_noop(stream=cur)
    e1.record(cur)
    torch.cuda.synchronize()
    wall = []
    for _ in range(50):
        t0 = time.perf_counter(); m.mori_noop(stream=cur); torch.cuda.synchronize(); wall.append(time.perf_counter() - t0)
    return {"device_us_per_call": 1e3 * e0.elapsed_time(e1) / reps,
            "host_launch_plus_sync_us": 1e6 * float(np.median(wall)),
            "what": "mori_noop: an empty kernel through the same ctypes binding, same stream"}


def _wall_us(call, reps=50):
    import torch
    ts = []
    for _ in range(reps):
        t0 = time.perf_counter(); call(); torch.cuda.synchronize(); ts.append(time.perf_counter() - t0)
    return 1e6 * float(np.median(ts))


def rank_partition_leg(with_oracle: bool, reps=200):
    """a1-a4 alone: device microseconds per call (CUDA events over `reps` back-to-back launches)
    and host wall-clock of one launch + sync, at cfg 2's n = 64 and cfg 5's n = 4096 (scores
    i.i.d. lognormal, sizes uniform, capacities that put the boundaries mid-ranking); the
    oracle's microseconds beside it when allowed (rank 0, N = 1)."""
    import torch
    from paper_2606_00866_b200 import binding
    pool = torch.zeros(2 * 4 * 8192, dtype=torch.uint8, device="cuda")
    m = binding.Mori(2, 2, 64, 16, pool, max_programs=4096)
    rng = np.random.default_rng(SEED)
    cur = torch.cuda.current_stream()
    out = {"floor": launch_floor(m, cur, reps)}
    for n in (64, 4096):
        iota = rng.lognormal(0.0, 1.0, n).astype(np.float32)
        kv = rng.integers(16, 513, n).astype(np.int32)
        prev = rng.integers(0, 3, n).astype(np.uint8)
        cg, cc = int(kv.sum() * 0.2), int(kv.sum() * 0.4)
        d = "cuda"
        t_i, t_s, t_p = (torch.from_numpy(x).to(d) for x in (iota, kv, prev))
        order = torch.empty(n, dtype=torch.int32, device=d); tier = torch.empty(n, dtype=torch.uint8, device=d)
        bounds = torch.empty(2, dtype=torch.int32, device=d); used = torch.empty(2, dtype=torch.int64, device=d)
        lists = torch.empty(5 * n, dtype=torch.int32, device=d); counts = torch.empty(5, dtype=torch.int32, device=d)

        def call():
            m.mori_rank_partition(n, t_i, t_s, t_p, cg, cc, order, tier, bounds, used, lists, counts, stream=cur)
        for _ in range(10):
            call()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(cur)
        for _ in range(reps):
            call()
        e1.record(cur)
        torch.cuda.synchronize()
        wall = []
        for _ in range(50):
            t0 = time.perf_counter(); call(); torch.cuda.synchronize(); wall.append(time.perf_counter() - t0)
        ent = {"device_us_per_call": 1e3 * e0.elapsed_time(e1) / reps,
               "host_launch_plus_sync_us": 1e6 * float(np.median(wall))}
        # NEXT-1: the sticky, status-aware policy mode on the same programs (GPU queue 1.5x over
        # its capacity so that victims are cut, CPU queue with room for some of them)
        fl = rng.integers(0, 8, n).astype(np.uint8)
        t_f = torch.from_numpy(fl).to(d)
        lazy = torch.empty(n, dtype=torch.uint8, device=d)
        scg = int(kv[prev == 0].sum() / 1.5)
        scc = int(kv[prev == 1].sum()) + int(kv[prev == 0].sum() * 0.2)

        def call_sticky():
            m.mori_sticky_rebalance(n, t_i, t_s, t_p, t_f, scg, scc, tier, lazy, used, lists, counts, stream=cur)
        for _ in range(10):
            call_sticky()
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(cur)
        for _ in range(reps):
            call_sticky()
        s1.record(cur)
        torch.cuda.synchronize()
        ent["sticky_device_us_per_call"] = 1e3 * s0.elapsed_time(s1) / reps
        ent["sticky_host_launch_plus_sync_us"] = _wall_us(call_sticky)
        # NEXT-2: Eq. (1) on the device: one tick's events (one completed cycle for a quarter of
        # the programs) + evaluation of all n scores
        me = max(1, n // 4)
        e_prog = rng.permutation(n)[:me].astype(np.int32)
        e_r, e_a = rng.lognormal(1.4, 0.5, me), rng.lognormal(1.0, 1.5, me)
        o_r, o_a = rng.lognormal(1.0, 0.5, n), rng.lognormal(2.0, 1.5, n)
        te = [torch.from_numpy(x).to(d) for x in (e_prog, np.zeros(me, np.uint8), e_r, e_a, o_r, o_a)]
        iota_d = torch.empty(n, dtype=torch.float32, device=d)

        def call_idl():
            m.mori_idleness_update(te[0], te[1], te[2], te[3], stream=cur)
            m.mori_idleness_eval(n, te[4], te[5], iota_d, stream=cur)
        for _ in range(10):
            call_idl()
        torch.cuda.synchronize()
        i0, i1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        i0.record(cur)
        for _ in range(reps):
            call_idl()
        i1.record(cur)
        torch.cuda.synchronize()
        ent["idleness_update_eval_device_us"] = 1e3 * i0.elapsed_time(i1) / reps
        # NEXT-4(i): Best-Fit-Decreasing of n Waiting-queue candidates across 8 replicas
        b_free = torch.from_numpy(np.full(8, int(kv.sum()) // 12, np.int64)).to(d)
        b_rep = torch.empty(n, dtype=torch.int32, device=d); b_left = torch.empty(8, dtype=torch.int64, device=d)

        def call_bfd():
            m.mori_bfd_assign(t_s, t_i, t_f, b_free, b_rep, b_left, stream=cur)
        for _ in range(5):
            call_bfd()
        torch.cuda.synchronize()
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b0.record(cur)
        for _ in range(50):
            call_bfd()
        b1.record(cur)
        torch.cuda.synchronize()
        ent["bfd_device_us_per_call"] = 1e3 * b0.elapsed_time(b1) / 50
        ent["bfd_host_launch_plus_sync_us"] = _wall_us(call_bfd, 20)
        fl_wall = out["floor"]["host_launch_plus_sync_us"]
        ent["floor_us"] = fl_wall
        ent["x_floor"] = {"rank_partition": ent["host_launch_plus_sync_us"] / fl_wall,
                          "sticky": ent["sticky_host_launch_plus_sync_us"] / fl_wall,
                          "bfd": ent["bfd_host_launch_plus_sync_us"] / fl_wall}
        if with_oracle:
            import oracle
            ts = []
            for _ in range(10):
                t0 = time.perf_counter(); oracle.bfd_assign(kv, iota, fl, np.full(8, int(kv.sum()) // 12)); ts.append(time.perf_counter() - t0)
            ent["bfd_oracle_us_1core"] = 1e6 * float(np.median(ts))
            trk = oracle.IdlenessTracker(n)
            ts = []
            for _ in range(20):
                t0 = time.perf_counter(); trk.update(e_prog, np.zeros(me, np.uint8), e_r, e_a); trk.eval(o_r, o_a)
                ts.append(time.perf_counter() - t0)
            ent["idleness_oracle_us_1core"] = 1e6 * float(np.median(ts))
            ts = []
            for _ in range(50):
                t0 = time.perf_counter(); oracle.rank_partition(iota, kv, prev, cg, cc); ts.append(time.perf_counter() - t0)
            ent["oracle_us_per_call_1core"] = 1e6 * float(np.median(ts))
            ts = []
            for _ in range(10):
                t0 = time.perf_counter(); oracle.sticky_rebalance(iota, kv, prev, fl, scg, scc); ts.append(time.perf_counter() - t0)
            ent["sticky_oracle_us_per_call_1core"] = 1e6 * float(np.median(ts))
        out[f"n{n}"] = ent
    m.close()
    return out


def eviction_leg(with_oracle: bool, n_pages=65536, n_programs=64, reps=50):
    """NEXT-3: typed eviction order of a 65 536-page pool (cfg 2's arena): device microseconds per
    call (15 kernels), and the oracle's qsort beside it."""
    import torch
    from paper_2606_00866_b200 import binding
    pool = torch.zeros(n_pages * 32, dtype=torch.uint8, device="cuda")       # 32-byte pages
    m = binding.Mori(1, 1, 8, 1, pool)
    rng = np.random.default_rng(SEED)
    owner = rng.integers(-1, n_programs, n_pages).astype(np.int32)
    ptier = rng.integers(0, 3, n_programs).astype(np.uint8)
    last = rng.integers(0, 200, n_pages).astype(np.uint32)                   # ticks
    d = "cuda"
    t_o, t_t = torch.from_numpy(owner).to(d), torch.from_numpy(ptier).to(d)
    t_l = torch.from_numpy(last.view(np.int32)).to(d)
    vic = torch.empty(n_pages, dtype=torch.int32, device=d); nres = torch.empty(1, dtype=torch.int32, device=d)
    cur = torch.cuda.current_stream()
    for _ in range(5):
        m.mori_eviction_order(binding.TIER_GPU, t_o, t_t, t_l, vic, nres, stream=cur)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(cur)
    for _ in range(reps):
        m.mori_eviction_order(binding.TIER_GPU, t_o, t_t, t_l, vic, nres, stream=cur)
    e1.record(cur)
    torch.cuda.synchronize()
    out = {"n_pages": n_pages, "device_us_per_call": 1e3 * e0.elapsed_time(e1) / reps}
    fl = launch_floor(m, cur)
    out["host_launch_plus_sync_us"] = _wall_us(lambda: m.mori_eviction_order(binding.TIER_GPU, t_o, t_t, t_l, vic, nres, stream=cur))
    out["floor_us"] = fl["host_launch_plus_sync_us"]
    out["floor_device_us_per_call"] = fl["device_us_per_call"]
    out["x_floor"] = out["host_launch_plus_sync_us"] / fl["host_launch_plus_sync_us"]
    # full-range 32-bit counters (five radix passes instead of two)
    t_l2 = torch.from_numpy(rng.integers(0, 2 ** 32, n_pages, dtype=np.uint64).astype(np.uint32).view(np.int32)).to(d)
    for _ in range(3):
        m.mori_eviction_order(binding.TIER_GPU, t_o, t_t, t_l2, vic, nres, stream=cur)
    torch.cuda.synchronize()
    e0.record(cur)
    for _ in range(reps):
        m.mori_eviction_order(binding.TIER_GPU, t_o, t_t, t_l2, vic, nres, stream=cur)
    e1.record(cur)
    torch.cuda.synchronize()
    out["device_us_per_call_full_range_counters"] = 1e3 * e0.elapsed_time(e1) / reps
    if with_oracle:
        import oracle
        ts = []
        for _ in range(5):
            t0 = time.perf_counter(); oracle.eviction_order(0, owner, ptier, last); ts.append(time.perf_counter() - t0)
        out["oracle_us_per_call_1core"] = 1e6 * float(np.median(ts))
    m.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=24)
    ap.add_argument("--warmup", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config, 1-based")
    ap.add_argument("--scale", type=int, default=0, help="0 = auto (1 when the pools fit)")
    ap.add_argument("--f-busy", type=float, default=None,
                    help="stationary busy fraction of the trace (cfg 3 sweeps 0.25 / 0.5 / 0.75; default: the config's)")
    ap.add_argument("--no-per-config", dest="per_config", action="store_false",
                    help="skip the per_config legs (every other BASELINE.json config after the headline one)")
    ap.add_argument("--per-config-steps", type=int, default=8, help="timed epochs of each per_config leg")
    ap.add_argument("--ref-threads", type=int, default=1, help="--impl reference: host threads of the oracle's movers")
    ap.add_argument("--path-demote", default="auto", choices=["auto", "zerocopy", "staged", "copyengine"])
    ap.add_argument("--path-promote", default="auto", choices=["auto", "zerocopy", "staged", "copyengine"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "ldst", "tma"])
    ap.add_argument("--staging-mib", type=int, default=0, help="0 = library default")
    ap.add_argument("--policy", default="partition", choices=["partition", "sticky"],
                    help="partition: re-partition every epoch (the hot path, default); sticky: the paper's "
                         "section-4.3.1 tier management (mori_sticky_rebalance)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="process-group backend for N > 1 (gloo + --device-index: exercise the N > 1 path on one GPU)")
    ap.add_argument("--device-index", type=int, default=-1, help="CUDA device to use instead of LOCAL_RANK")
    ap.add_argument("--verbose", action="store_true", help="per-step lines on stderr")
    ap.add_argument("--timeline", default=None, metavar="FILE",
                    help="write the per-stream event timeline of every timed step of the headline config to FILE (JSON)")
    ap.add_argument("--leg", default=None, choices=["copy_sweep", "three_tier"],
                    help="run one auxiliary measurement leg instead of the bench line (copy_sweep: the gather/scatter "
                         "kernel alone and in-step for several ring geometries; profiles/ cites it)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-gather-leg", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.leg == "copy_sweep":
        copy_kernel_sweep(args)
    elif args.leg == "three_tier":
        three_tier_leg(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
