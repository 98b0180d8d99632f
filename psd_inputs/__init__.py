"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests/bench.

This package holds NONE of the method's arithmetic (no tets, no clipping, no deposit):
it only makes particle positions.  Neither oracle/ nor paper_1612_09491_b200/ is
imported here.  Recipe and citations: DESIGN.md "Input recipe"; PAPER.md:165 (the
paper's Dark Sky snapshots, which these stand in for) and PAPER.md:175 (its analytic
weak-scaling workload).
"""
from .zeldovich import (CONFIGS, config_positions, jittered_lattice, lattice, sha256_of,
                        splitmix64, zeldovich_positions)

__all__ = ["CONFIGS", "config_positions", "jittered_lattice", "lattice", "sha256_of",
           "splitmix64", "zeldovich_positions"]
