"""B200-native MORI hot path: idleness rank/partition + paged-KV demote/promote (sm_100a).

``paper_2606_00866_b200.binding`` is the ctypes binding over ``libmori.so`` (C ABI declared in
``include/mori.h``); ``paper_2606_00866_b200.workload`` makes the seeded synthetic inputs.
There is no CPU fallback: using the binding without the built CUDA library raises.
"""
__all__ = ["binding", "workload", "build", "harness", "replicas"]
