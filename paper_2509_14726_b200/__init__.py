"""B200-native MPPI hot path (arXiv 2509.14726): C-ABI library `libmppi` + thin Python binding.

Importing the package does not load the CUDA library; `paper_2509_14726_b200.binding` does, and
fails loudly when it is missing.  `workloads` (seeded synthetic inputs) is pure numpy.
"""
__all__ = ["binding", "workloads", "build"]
