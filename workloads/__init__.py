"""Seeded synthetic input generators for the SDM coalescence hot path.

This module is shared by the CPU oracle's tests and by the CUDA path's tests/bench and
holds NONE of the method's arithmetic (no Philox, no pairing, no probability, no update):
it only builds initial states (xi, v, cell_id) and the scalar parameters of each workload.
The recipes follow BASELINE.json `configs` and SURVEY.md section 8(d); DESIGN.md restates them.
"""
from .configs import (  # noqa: F401
    Workload,
    golovin_box,
    gravitational_box,
    grid_poisson,
    grid_uniform,
    grid_small_multiplicity,
    make,
    spectrum_bins,
    V_MEAN_BOX,
    V_MEAN_C5,
)
