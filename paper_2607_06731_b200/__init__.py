"""paper_2607_06731_b200 — B200-native Beagle scoring (batched colony fitness evaluation).

The product is the C-ABI library built from csrc/ (include/beagle.h); `api` is its thin ctypes
binding (argument marshalling only). `colonies` is the seeded input generator of the host harness.
"""
__all__ = ["api", "colonies"]
