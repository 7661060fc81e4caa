"""N > 1: independent replicas, no data-path collective.

The paper's placement is per replica: "Each inference engine replica maintains its own GPU and CPU
queues" and every replica "appl[ies] the same rule of filling from the busiest end of the
ranking until local capacity is reached".  So rank r runs the whole hot path on its own
programs (its own seeded trace), its own pool and its own pinned arena over its own host link;
nothing of the KV path crosses NVLink.  The cross-rank steps are bookkeeping: the job's time is
the slowest rank's, its work the sum (one all-reduce of a few float64), and -- for the shared
Waiting queue of P:L180 -- an all-gather of each replica's free capacity, through
``torch.distributed`` (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import Sequence, Tuple


def env_rank() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) as torchrun exports them; (0, 1, 0) without a launcher."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_seed(seed: int, rank: int) -> int:
    """Every replica draws its own programs: a distinct trace / page-table stream per rank."""
    return seed + rank


def aggregate(times_s: Sequence[float], sums: Sequence[float], device="cpu"):
    """-> (max over ranks of every entry of ``times_s``, sum over ranks of every entry of
    ``sums``).  A no-op without an initialised process group (single replica)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(x) for x in times_s], [float(x) for x in sums]
    t = torch.tensor(list(times_s), dtype=torch.float64, device=device)
    s = torch.tensor(list(sums), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return t.tolist(), s.tolist()


def gather_free_capacity(free_local_pages: int, device="cpu"):
    """The one piece of cross-replica data of the paper's design: every replica's free GPU pages,
    all-gathered so that each replica can run the same Best-Fit-Decreasing packing of the shared
    Waiting queue (``mori_bfd_assign``).  -> int64 tensor [world] on ``device``
    (stays on the GPU under NCCL, so it feeds the kernel without a host round trip)."""
    import torch
    import torch.distributed as dist
    mine = torch.tensor([int(free_local_pages)], dtype=torch.int64, device=device)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return mine
    parts = [torch.empty_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, mine)
    return torch.cat(parts)


def throughput_gbps(times_s: Sequence[float], bytes_moved: Sequence[float], device="cpu") -> float:
    """Whole-job GB/s: bytes all replicas moved / the slowest replica's time."""
    (t,), (b,) = aggregate([sum(times_s)], [sum(bytes_moved)], device)
    return b / t / 1e9 if t > 0 else 0.0
