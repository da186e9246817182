"""CPU oracle for the gamma-index hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_1012_1900_b200.
"""
from .gamma_oracle import (  # noqa: F401
    build,
    gamma,
    num_threads,
    simplex_distance,
    simplex_distance_ju,
)
