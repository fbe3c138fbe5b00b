"""Seeded synthetic inputs for the PPM hot path (shared by the oracle tests and the CUDA path).

Holds NONE of the method's arithmetic: only grids, parameter vectors, the synthetic atmosphere
table, the synthetic response and helpers to pack parameter vectors.  See DESIGN.md "Input recipe".
"""
from .workloads import *  # noqa: F401,F403
