"""B200-native quadtree lattice-Boltzmann hot path (after arXiv 2504.04465).

`paper_2504_04465_b200.lbm` is the thin binding over the C-ABI CUDA library (it fails loudly if the
library is not built); `paper_2504_04465_b200.workloads` holds the seeded input generators.
Nothing is imported eagerly so that the input generators stay usable without the CUDA library.
"""
__all__ = ["lbm", "workloads"]
