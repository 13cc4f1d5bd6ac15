"""Seeded, synthetic input generators and plain data containers.

This package serves both the CPU oracle (`oracle/`) and the CUDA library
(`paper_1309_5571_b200/`).  It holds NONE of the method's arithmetic: no
Kronecker products, no projections, no eigen-solvers -- only containers for
"operators stored as dense blocks per symmetry sector" (Sec. 4.1)
and the seeded random recipes of DESIGN.md ("Input recipe").
"""
from .problem import Sectors, BlockOp, Problem
from .synthetic import (heisenberg_synthetic, hubbard_synthetic, sector_profile,
                        random_vector, vector_seed, CONFIGS, make_config,
                        SimpleBlock, heisenberg_block_synthetic)

__all__ = ["Sectors", "BlockOp", "Problem", "heisenberg_synthetic", "hubbard_synthetic",
           "sector_profile", "random_vector", "vector_seed", "CONFIGS", "make_config",
           "SimpleBlock", "heisenberg_block_synthetic"]
