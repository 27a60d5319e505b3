"""bfsc — B200-native delta + patched-FOR codec for BFS frontier traffic (arxiv 1704.00513).

The product is the C-ABI library built from csrc/ (include/bfsc.h) and the thin binding in
`binding.py`; `workloads/` holds the seeded input generators. Importing this package does
not load the CUDA library (so it imports on a CPU-only box); the first call does, and fails
loudly if the library is missing — there is no CPU fallback.
"""
__all__ = ["binding", "workloads"]
