"""Seeded synthetic inputs for the Chebyshev-filter hot path (shared by the oracle tests and the CUDA path).

This package holds NONE of the method's arithmetic: no shape functions, no quadrature weights, no cell
matrices, no recurrence.  It only produces inputs: mesh connectivity, vertex coordinates, and *samples* of
the synthetic potential / projector functions at the Gauss-point positions, plus the random vector block.
"""
from .generate import (CONFIGS, ConfigSpec, Workload, make_mesh, make_workload, gauss_points_physical,
                       random_block, load_bounds)

__all__ = ["CONFIGS", "ConfigSpec", "Workload", "make_mesh", "make_workload", "gauss_points_physical",
           "random_block", "load_bounds"]
