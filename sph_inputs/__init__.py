"""Seeded synthetic SPH inputs shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no packing, no kernel
function, no neighbour sums, no cell/task building).  It only draws particles
with a counter-based generator and writes them into the canonical 128-byte AoS
record that both sides accept as their input format (BASELINE.json:configs[0]).

The paper's own datasets (Gresho256, Eagle25) are not
available here; these generators stand in for their shape ("Input
recipe").
"""
from .format import PART_DTYPE, FIELDS, FIELD_NCOMP, field_id  # noqa: F401
from .generators import (  # noqa: F401
    splitmix64, uniform01, normal01,
    config0, config1, config2_positions, config3, config4,
    jittered_lattice, clumpy_mixture, mixture_density, eagle_like, eagle_like_counts, synthetic_trace,
)
