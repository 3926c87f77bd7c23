"""B200-native combinatorial-summation (CoS) evaluation of connected Feynman-diagram sums.

Public API (thin ctypes binding over the C-ABI library `libcos_b200.so`, see include/cos.h):
    from paper_2501_00675_b200 import api      # cos_create, cos_build_G, cos_eval_connected, ...
    from paper_2501_00675_b200 import workloads  # seeded synthetic inputs (numpy only)
"""
__all__ = ["api", "workloads"]
