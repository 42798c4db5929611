"""paper_2004_04334_b200 — B200-native pixel local reconstruction behind an acquire/produce C-ABI.

The product is ``csrc/`` (sm_100a CUDA kernels + the ``pr_*`` C-ABI of ``include/pixreco.h``) and
the thin ctypes binding in :mod:`paper_2004_04334_b200.pixreco`.  ``workloads`` is the seeded
input generator (no method arithmetic).  Nothing here imports ``oracle/``.
"""
__all__ = ["pixreco", "workloads"]
