"""Seeded synthetic input generators (images, (u, v), weights, noise) shared by the oracle's tests, the
CUDA path's tests, bench.py and smoke().  A module of its own: it holds none of the method's arithmetic
and imports neither oracle/ nor paper_1903_04502_b200/ (numpy only)."""
from . import synth  # noqa: F401
