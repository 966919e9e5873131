"""Seeded synthetic input generators shared by the oracle-side tests and the CUDA-side runs.
Holds none of the method's arithmetic."""
from . import rng, configs  # noqa: F401
