"""CPU oracle for the gamma-index hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_1012_1900_b200.
"""
from .gamma_oracle import (  # noqa: F401
    gamma,
    num_threads,
    simplex_distance,
    simplex_distance_ju,
)
from .gamma_oracle import build as _build_same_grid
from .gamma_general_oracle import build as _build_general
from .gamma_general_oracle import gamma_general  # noqa: F401


def build(force: bool = False):
    """Compile every C file of the oracle (gamma_oracle.c, gamma_general_oracle.c) with gcc."""
    _build_general(force)
    return _build_same_grid(force)
