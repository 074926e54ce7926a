"""Seeded synthetic inputs for the H_eff*psi hot path (shared by the oracle, the tests and bench.py).

This package only *draws* inputs: sector tables, operator-block descriptors, operator entries,
coefficients and wavefunction entries.  It contains none of the method's arithmetic (no contraction,
no flop model, no scheduling) and imports neither ``oracle`` nor ``paper_2407_07411_b200``.

The recipes restate SURVEY.md section 8(d) / DESIGN.md "Input recipe"; they stand in for the paper's
real-molecule workloads (F2 / N2 / FeMoco / P450), whose integral files do not exist here.
"""
from .configs import (CONFIG_NAMES, OPBLOCK_DTYPE, Problem, make_problem, make_psi, make_shard, term_chunk, config_params,
                      custom_problem)
from .hubbard import hubbard_two_block_problem
from .site import make_isometries, pack_isometries, proportional_chi

__all__ = ["CONFIG_NAMES", "OPBLOCK_DTYPE", "Problem", "make_problem", "make_psi", "config_params",
           "custom_problem", "make_shard", "term_chunk", "hubbard_two_block_problem", "make_isometries", "pack_isometries", "proportional_chi"]
