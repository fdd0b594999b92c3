"""B200-native TPC track reconstruction hot path (arXiv 2106.03636, BASELINE.json north_star).

Importing the package is cheap and CPU-safe; the CUDA library is loaded on first use by
`paper_2106_03636_b200.binding` and fails loudly when it is missing (there is no CPU fallback).
"""
__version__ = "0.1.0"
