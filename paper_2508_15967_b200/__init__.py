"""B200-native batched RF ray tracing (arxiv/paper_2508_15967's demonstration problem).

``paper_2508_15967_b200.binding`` -- thin ctypes binding of the C-ABI library (include/rt.h); every step of
                                     the hot path runs in the library's sm_100a CUDA kernels.
``paper_2508_15967_b200.inputs``  -- seeded synthetic workloads (no method arithmetic; shared with the oracle's tests).
"""

__all__ = ["binding", "inputs"]
