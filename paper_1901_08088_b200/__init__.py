"""qbvh — quantized-BVH neighbor lists (Howard et al., arXiv:1901.08088) for NVIDIA B200 (sm_100a).

The product is the C-ABI library ``libqbvh.so`` (``include/qbvh.h``) built from
``csrc/``; :mod:`paper_1901_08088_b200.qbvh` is the thin ctypes binding with the
same names.  :mod:`paper_1901_08088_b200.workloads` holds the seeded synthetic
input generators (no method arithmetic).  Nothing here imports ``oracle/``.
"""
__all__ = ["qbvh", "workloads", "build"]
