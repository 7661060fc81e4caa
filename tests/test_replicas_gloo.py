"""N > 1 host logic on CPU: two gloo ranks, each an independent replica (own seeded programs,
own placement), aggregated the way bench.py does -- max of times, sum of bytes."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _replica_epochs(rank, epochs=6):
    """Placement + planned migration of one replica (oracle placement: this is a CPU test)."""
    import oracle
    from paper_2606_00866_b200 import replicas, workload as W
    cfg = W.get_config(1)
    sim = W.Sim(cfg, replicas.replica_seed(866, rank))
    moved, tiers = 0, []
    for _ in range(epochs):
        plan = sim.begin_epoch()
        res = oracle.rank_partition(plan.iota, plan.kv_pages, plan.prev_tier, cfg.cap_gpu_pages, cfg.cap_cpu_pages)
        sim.apply_placement(res["tier"], res["lists"])
        sim.end_epoch()
        moved += (plan.demote_pages + plan.promote_pages) * cfg.shape.page_bytes
        tiers.append(res["tier"].copy())
    return moved, tiers


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2606_00866_b200 import replicas
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert replicas.env_rank() == (rank, world, rank)
    moved, tiers = _replica_epochs(rank)
    t_local = 0.25 * (rank + 1)                      # rank 1 is the slow one
    (t,), (b, n) = replicas.aggregate([t_local], [moved, 1.0])
    gbps = replicas.throughput_gbps([t_local], [moved])
    # shared Waiting queue: all-gather the replicas' free capacity, pack with the oracle's BFD
    import numpy as np, oracle
    free = replicas.gather_free_capacity(100 * (rank + 1) + 7).numpy()
    rng = np.random.default_rng(12)                                   # the same queue on every rank
    size = rng.integers(1, 60, 25).astype(np.int32)
    iota = rng.random(25).astype(np.float32)
    flags = (2 | (rng.integers(0, 2, 25) * 4)).astype(np.uint8)
    rep, left = oracle.bfd_assign(size, iota, flags, free)
    q.put((rank, t, b, n, gbps, moved, [x.tolist() for x in tiers], free.tolist(), rep.tolist(), left.tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_aggregate_like_the_bench():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    sys.path.insert(0, ROOT)
    want = [_replica_epochs(r) for r in range(2)]
    assert got[0][7] == got[1][7] == [107, 207]                      # every rank sees every capacity
    assert got[0][8] == got[1][8] and got[0][9] == got[1][9]          # ... and packs identically
    assert {0, 1} <= set(got[0][8])                                   # both replicas admit someone
    for r, (rank, t, b, n, gbps, moved, tiers, *_rest) in enumerate(got):
        assert rank == r
        assert moved == want[r][0]                                  # replicas are deterministic
        assert tiers == [x.tolist() for x in want[r][1]]
        assert t == 0.5 and n == 2.0                                # max over ranks / all ranks counted
        assert b == want[0][0] + want[1][0]                         # bytes sum over replicas
        assert np.isclose(gbps, b / 0.5 / 1e9)
    # the two replicas really hold different programs
    assert [x.tolist() for x in want[0][1]] != [x.tolist() for x in want[1][1]] or want[0][0] != want[1][0]


def test_single_replica_aggregate_is_identity():
    from paper_2606_00866_b200 import replicas
    assert replicas.aggregate([1.5, 2.0], [3.0]) == ([1.5, 2.0], [3.0])
    assert replicas.throughput_gbps([1.0, 1.0], [4e9]) == 2.0
    assert replicas.replica_seed(866, 3) == 869
    assert replicas.gather_free_capacity(42).tolist() == [42]
