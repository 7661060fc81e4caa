"""CPU oracle for the MORI hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2606_00866_b200`` and neither imports the other.

Two independent statements of the same definitions live here:

* ``oracle.c``      plain C (qsort + while loops + memcpy), loaded through ctypes by ``c_oracle``;
* ``oracle_np.py``  numpy restatement (stable argsort, cumsum, searchsorted, fancy indexing).

Citations ``P:Lnnn`` are lines of the paper text.
"""
from .c_oracle import (build, rank_partition, bruteforce_partition, demote, promote,  # noqa: F401
                       sticky_rebalance, IdlenessTracker, eviction_order, bfd_assign, rank_partition_tiers, move_slots, lib_path)
from . import oracle_np  # noqa: F401
