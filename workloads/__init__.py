"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs[0..4]).

This module serves BOTH the oracle and the CUDA path and therefore holds none
of the method's arithmetic: no eikonal solve, no weighting, no interpolation,
no back projection.  It builds geometry (grid, speed-of-sound map, sensors,
ROI) and, GIVEN a travel-time table computed elsewhere, synthesises sensor
traces.  The recipe is documented in DESIGN.md ("Input recipe"); it stands in
for the CT-derived monkey-skull model and k-Wave traces of PAPER.md:73, which
are not available.
"""
from .configs import (Geometry, CONFIG_NAMES, make_geometry, make_absorbers, make_traces,
                      frame_seed, BASE_SEED)

__all__ = ["Geometry", "CONFIG_NAMES", "make_geometry", "make_absorbers", "make_traces",
           "frame_seed", "BASE_SEED"]
