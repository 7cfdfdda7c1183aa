"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NO arithmetic of the transit model itself (no grid, no weights, no orbit, no
lens area, no flux): it only draws parameter vectors and limb-darkening coefficients and samples
the caller-side LD law on a mu grid that the caller passes in (the oracle's own grid for the
oracle, ``rr_get_mu`` for the CUDA library).  It imports neither ``oracle`` nor the product
package.  The recipe is stated in DESIGN.md section 4 and follows BASELINE.json ``configs``.
"""
from .configs import (ModelConfig, Workload, make_workload, sample_profile, CONFIG_NAMES,
                      paper_dummy_example)

__all__ = ["ModelConfig", "Workload", "make_workload", "sample_profile", "CONFIG_NAMES",
           "paper_dummy_example"]
