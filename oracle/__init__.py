"""CPU oracle for the log-polar thin-disk potential -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_2409_02294_b200.
"""
from .polar_oracle import (  # noqa: F401
    build, grid, potential_o0, potential_o0_targets, potential_o1, potential_o1_rings,
    num_threads, ext_o0, ext_o0_targets, ext_o1, ext_o1_rings, SOFT_SYMMETRIC, SOFT_FIELD, SOFT_SOURCE,
    cart_potential, cart_potential_targets, cart_self_constant,
)
from .definition_numpy import potential_definition_numpy  # noqa: F401
from . import nested_oracle  # noqa: F401  (NEXT-3: nested meshes, step-by-step algorithm)
