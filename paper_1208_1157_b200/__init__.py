"""B200-native ensemble n-body step loop (Hermite + MVS, FP64) after Swarm-NG, arxiv 1208.1157.

``paper_1208_1157_b200.ens``        thin ctypes binding over the C-ABI library ``libens.so`` (include/ens.h)
``paper_1208_1157_b200.workloads``  seeded synthetic ensembles (no method arithmetic)
``paper_1208_1157_b200.build``      in-tree nvcc build of ``csrc/`` for sm_100a

There is no CPU fallback: every entry point of ``ens`` raises if ``libens.so`` is missing or CUDA fails.
"""
__all__ = ["ens", "workloads", "build"]
