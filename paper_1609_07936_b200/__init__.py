"""sail-b200: B200-native hot path of SAIL (arXiv 1609.07936) — population-parallel Monte Carlo anneal.

The product is the C-ABI shared library `libsail_b200.so` (declared in include/sail.h, built from
paper_1609_07936_b200/csrc/*.cu for sm_100a) plus the thin ctypes binding in `binding.py`.
Importing this package does not load the library; the first call through `binding` does and fails
loudly if it is missing.  There is no CPU fallback.
"""
__all__ = ["binding", "workloads", "build"]
