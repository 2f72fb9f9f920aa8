"""paper_1901_01895_b200 — B200-native RK4IP propagator for the multimode Manakov/NLSE (arXiv 1901.01895).

The product is the C-ABI CUDA library (include/mmf.h, csrc/) and this thin binding.  `workloads` holds the seeded
synthetic inputs; it is importable without a GPU.  Nothing here imports the CPU oracle.
"""
__all__ = ["binding", "workloads", "build"]
