"""Seeded synthetic workloads shared by the CPU oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no Wick sums, no DAG, no
interpolation).  It only produces *inputs*:

  * the five BASELINE.json configurations (`CONFIGS`),
  * free-propagator lookup tables g_sigma(r, tau) on `n_tau` imaginary-time
    nodes (exact k-sum; Eq. 47-48, conventions SURVEY.md
    section 8(c) G16-G19),
  * seeded Monte-Carlo-like configurations (vertex sites, sublattices, times), uniform or clustered (stress input),
  * plain random propagator matrices for unit tests.

Both `oracle/` and `paper_2507_12349_b200/` consume these arrays; neither
imports the other.  The inputs stand in for the paper's Monte-Carlo
configurations (32x32 lattices, beta<=10), which are
not available.
"""
from .configs import CONFIGS, Workload, get_config
from .tables import build_table, PropTable
from .draws import draw_clustered_vertices, draw_vertices, random_matrices

__all__ = [
    "CONFIGS", "Workload", "get_config", "build_table", "PropTable",
    "draw_vertices", "draw_clustered_vertices", "random_matrices",
]
