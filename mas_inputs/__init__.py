"""Seeded synthetic inputs (meshes, coefficient fields, right-hand sides) for the MAS PCG path.

Shared by the oracle's tests, the CUDA parity tests and bench.py.  Holds none of the method's
arithmetic; see grids.py and configs.py.
"""
from . import grids, configs  # noqa: F401
