"""Seeded synthetic input generators (shared by the oracle tests and the CUDA path)."""
from . import phantom  # noqa: F401
