"""paper_1805_11991_b200 -- B200-native batched naive Hasse-Weil counts (arXiv 1805.11991).

`workloads` (numpy only) holds the seeded input generators; `hec` is the thin ctypes
binding of the C-ABI library libhec.so (include/hec.h).  Importing the package does not
load the CUDA library; the first call into `hec` does, and fails loudly if it is missing.
"""
__all__ = ["workloads", "hec"]
