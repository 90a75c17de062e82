"""Bin-edge arrays (inputs to both the oracle and the CUDA path).

PAPER.md:103 names three presets -- even, natural-log and log10 spacing between a
user-chosen low and high limit -- without formulas.  Natural-log and log10 spacing
give the same geometric edges (reading R5); so two helpers suffice.
Edges are data: both sides bin against exactly the doubles returned here.
"""
from __future__ import annotations

import math

import numpy as np


def log_theta_edges_deg(theta_min_deg: float, theta_max_deg: float, nbins: int) -> np.ndarray:
    """theta_k = theta_min * (theta_max/theta_min)**(k/nbins), k = 0..nbins (degrees)."""
    if not (0.0 < theta_min_deg < theta_max_deg <= 180.0) or nbins < 1:
        raise ValueError("need 0 < theta_min < theta_max <= 180 and nbins >= 1")
    ratio = theta_max_deg / theta_min_deg
    e = np.array([theta_min_deg * ratio ** (k / nbins) for k in range(nbins + 1)], dtype=np.float64)
    e[0], e[-1] = theta_min_deg, theta_max_deg
    return e


def linear_theta_edges_deg(theta_min_deg: float, theta_max_deg: float, nbins: int) -> np.ndarray:
    """Evenly spaced bins (PAPER.md:103 'evenly spaced bins')."""
    if not (0.0 <= theta_min_deg < theta_max_deg <= 180.0) or nbins < 1:
        raise ValueError("need 0 <= theta_min < theta_max <= 180 and nbins >= 1")
    e = np.array([theta_min_deg + (theta_max_deg - theta_min_deg) * k / nbins for k in range(nbins + 1)],
                 dtype=np.float64)
    e[0], e[-1] = theta_min_deg, theta_max_deg
    return e


def cos_edges_from_theta_deg(theta_edges_deg) -> np.ndarray:
    """Ascending theta edges (deg) -> strictly descending cosine edges.

    theta = 0 maps to exactly 1.0 and theta = 180 to exactly -1.0, so that a range
    reaching the pole really contains every pair (the pair cosine is clamped to
    [-1, 1]).  Raises if two edges collapse onto the same double.
    """
    t = np.asarray(theta_edges_deg, dtype=np.float64)
    out = np.empty_like(t)
    for k, th in enumerate(t):
        if th == 0.0:
            out[k] = 1.0
        elif th == 180.0:
            out[k] = -1.0
        else:
            out[k] = math.cos(math.radians(float(th)))
    if not np.all(np.diff(out) < 0):
        raise ValueError("cosine edges are not strictly descending (bins too fine for fp64)")
    return out
