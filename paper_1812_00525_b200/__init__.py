"""paper_1812_00525_b200 -- B200-native (sm_100a, FP64) hot path of CLTx (arxiv 1812.00525).

The product is the C-ABI library ``libclt.so`` (``include/clt.h``; CUDA sources in ``csrc/``);
``clt`` is the thin ctypes binding with the same names; ``inputs`` is the seeded synthetic workload
recipe shared with the tests of the CPU oracle.  Nothing here imports ``oracle``.
"""
__all__ = ["inputs", "clt", "slab", "replicas", "build"]
