"""Seeded synthetic inputs shared by the oracle, the CUDA path, the tests and bench.py.

This package holds NONE of the method's arithmetic (no unit vectors, no pair
cosines, no binning, no estimator): it only draws (RA, Dec[, weight]) catalogues
and writes bin-edge arrays.  Both sides receive the same arrays as inputs.

The catalogues stand in for the paper's unpublished N-body mock (PAPER.md:111-113:
clustered galaxies + a "flat" random catalogue over the same footprint); the five
configurations are BASELINE.json's.  Recipe: DESIGN.md "Synthetic inputs".
"""
from .bins import cos_edges_from_theta_deg, log_theta_edges_deg, linear_theta_edges_deg
from .catalogs import full_sky, lognormal_weights, neyman_scott, uniform_patch
from .configs import CONFIGS, make_config

__all__ = [
    "cos_edges_from_theta_deg", "log_theta_edges_deg", "linear_theta_edges_deg",
    "full_sky", "lognormal_weights", "neyman_scott", "uniform_patch",
    "CONFIGS", "make_config",
]
