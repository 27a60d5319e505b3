"""Seeded synthetic inputs shared by the tests, bench.py and smoke(). Holds none of the
codec's arithmetic; imports neither the CUDA binding nor the oracle."""
from . import rng, streams, rmat  # noqa: F401
