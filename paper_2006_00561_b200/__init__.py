"""B200-native population-annealing hot path (arxiv 2006.00561): thin ctypes binding over libpa_b200.so.

Importing the package does not load the CUDA library; `paper_2006_00561_b200.binding` does, and fails loudly
if it has not been built (there is no CPU fallback)."""
__all__ = ["inputs"]
