"""paper_2111_14999_b200 -- B200-native (sm_100a) el-ph Wannier->Bloch |g|^2 hot path
of Phoebe (arXiv 2111.14999): hand-written CUDA kernels behind a small C ABI
(include/phoebe_elph.h), a thin ctypes binding, and the seeded workload generator.

    from paper_2111_14999_b200 import binding, workloads, harness
"""
__all__ = ["binding", "workloads", "harness", "build"]
