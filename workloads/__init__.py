"""Seeded synthetic inputs for the UGKS step: problem descriptions and initial states.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's tests /
bench.  It holds plain data and the input recipe of DESIGN.md ("Input recipe"), none of the
method's arithmetic (no reconstruction, moments, fluxes or updates).  The one formula here
is the Maxwellian used to *draw* an initial f from seeded primitive fields, Eq. (1).
"""
from .channel import (BC_FIXED, BC_PERIODIC, BC_WALL, CONFIGS, Problem, channel_config,  # noqa: F401
                      initial_state, maxwellian_field, paper_mesh, periodic_box, trapezoid_grid, smooth_noise)
