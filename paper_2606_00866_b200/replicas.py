"""N > 1: independent replicas, no data-path collective.

The paper's placement is per replica: "Each inference engine replica maintains its own GPU and CPU
queues" and every replica "appl[ies] the same rule of filling from the busiest end of the
ranking until local capacity is reached".  So rank r runs the whole hot path on its own
programs (its own seeded trace), its own pool and its own pinned arena over its own host link;
nothing of the KV path crosses NVLink.  The only cross-rank step is the bookkeeping below: the
job's time is the slowest rank's, its work the sum -- one all-reduce of a few float64 through
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


def throughput_gbps(times_s: Sequence[float], bytes_moved: Sequence[float], device="cpu") -> float:
    """Whole-job GB/s: bytes all replicas moved / the slowest replica's time."""
    (t,), (b,) = aggregate([sum(times_s)], [sum(bytes_moved)], device)
    return b / t / 1e9 if t > 0 else 0.0
