"""B200-native per-cell exponential drag update (arXiv 2509.25347): thin Python binding over the C-ABI library.

Importing the package does not load CUDA; `paper_2509_25347_b200.binding` loads `libdg.so` and fails loudly
when it is missing.  `paper_2509_25347_b200.workloads` holds the seeded synthetic input generators only.
"""
__all__ = ["binding", "workloads", "build"]
