"""CPU oracle for the Abacus near-field force (arXiv:1810.02916).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It shares no code with
``paper_1810_02916_b200`` (the CUDA path) and neither imports the other.
"""
from .nf_oracle import (  # noqa: F401
    build,
    keys,
    bin_particles,
    forces,
    cell_amax,
    kick_drift,
    cell_vrms,
    timestep_terms,
    interactions,
    spline_over_r,
    plummer_over_r,
    max_threads,
    parity_error,
)
from . import nf_tree  # noqa: F401,E402  (tree near field for dense cells)
from .nf_tree import forces_tree  # noqa: F401,E402
