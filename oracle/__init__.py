"""CPU oracle for the CoS / SB-CoS connected sums (arxiv 2507.12349).

TEST INFRASTRUCTURE ONLY — see oracle/cos_oracle.c for the header.  Nothing under
paper_2507_12349_b200/ imports this package, and this package imports nothing from it.
"""
from .cos_oracle import (  # noqa: F401
    build_oracle, o1_connected, o1_all_subsets, o2a_twospin, o2b_polynomial,
    o3_alg3, o3_uniform, connected_reference, tabulate_reference, subset_blocks, flux_weights,
)
