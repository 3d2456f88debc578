"""Seeded synthetic inputs shaped like the paper's workloads.

This package is the ONLY code shared by the CUDA path's tests/bench and the CPU
oracle.  It holds none of the method's arithmetic (no stencil, no operator, no
LSQR): it builds velocity models, point-source right-hand sides, receiver node
lists and random data, in float64, and rounds ONCE to float32 / complex64
(reading C-14).  Both sides consume the rounded arrays.
"""
from .configs import Workload, make, CONFIG_NAMES, column_range  # noqa: F401
