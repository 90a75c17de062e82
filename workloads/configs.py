"""The five BASELINE.json configurations as seeded synthetic catalogues.

make_config(name, scale) draws data + random catalogues and the bin edges.  scale
< 1 shrinks the point (and parent) counts on the same footprint, for the parity
cases the CPU oracle must finish in seconds; scale = 1 is the configuration as
BASELINE.json states it.  Seeds: data / random = 1/2, 11/12, 21/22, 31/32 (weights
33/34), 41/42.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

from .bins import cos_edges_from_theta_deg, log_theta_edges_deg
from .catalogs import lognormal_weights, neyman_scott, uniform_patch


def _band_for_area(area_deg2: float, ra_width_deg: float) -> float:
    """Half-height (deg) of the Dec band symmetric about the equator whose area over
    ra_width_deg of RA is area_deg2:  area = ra_width * (180/pi) * 2 sin(dec_max)."""
    s = area_deg2 / (ra_width_deg * (180.0 / math.pi) * 2.0)
    return math.degrees(math.asin(s))


CONFIGS = {
    # name: n_data, n_random, RA range, Dec range, bins (theta_min_deg, theta_max_deg, nbins), clustering, weights
    "tiny": dict(n_d=10_000, n_r=10_000, ra=(0.0, 10.0), dec=(-5.0, 5.0),
                 bins=(1.0 / 60.0, 5.0, 20), cluster=None, seeds=(1, 2), weights=None),
    "clustered_patch": dict(n_d=200_000, n_r=200_000, ra=(0.0, 20.0), dec=(-10.0, 10.0),
                            bins=(0.5 / 60.0, 10.0, 25),
                            cluster=dict(n_parents=10_000, sigma_arcmin=3.0, children="fixed"),
                            seeds=(11, 12), weights=None),
    "survey_scale": dict(n_d=1_000_000, n_r=2_000_000, ra=(0.0, 40.0),
                         dec=(-_band_for_area(1000.0, 40.0), _band_for_area(1000.0, 40.0)),
                         bins=(0.1 / 60.0, 3.0, 30),
                         cluster=dict(n_parents=50_000, sigma_arcmin=5.0, children="poisson"),
                         seeds=(21, 22), weights=None),
    "full_sky": dict(n_d=1_000_000, n_r=1_000_000, ra=(0.0, 360.0), dec=(-90.0, 90.0),
                     bins=(1.0 / 60.0, 180.0, 40), cluster=None, seeds=(31, 32), weights=(33, 34)),
    "pruning_stress": dict(n_d=8_000_000, n_r=8_000_000, ra=(0.0, 360.0),
                           dec=(-_band_for_area(5000.0, 360.0), _band_for_area(5000.0, 360.0)),
                           bins=(0.2 / 60.0, 1.0, 15),
                           cluster=dict(n_parents=400_000, sigma_arcmin=2.0, children="poisson", wrap_ra=True),
                           seeds=(41, 42), weights=None),
}


@dataclass
class Workload:
    name: str
    scale: float
    ra_d: np.ndarray
    dec_d: np.ndarray
    ra_r: np.ndarray
    dec_r: np.ndarray
    theta_edges_deg: np.ndarray
    cos_edges: np.ndarray
    w_d: np.ndarray | None = None
    w_r: np.ndarray | None = None
    meta: dict = field(default_factory=dict)

    @property
    def n_d(self) -> int:
        return int(self.ra_d.size)

    @property
    def n_r(self) -> int:
        return int(self.ra_r.size)

    @property
    def nbins(self) -> int:
        return int(self.cos_edges.size - 1)

    @property
    def nominal_pairs(self) -> int:
        """DD + DR + RR pairs: n_d(n_d-1)/2 + n_d n_r + n_r(n_r-1)/2."""
        return self.n_d * (self.n_d - 1) // 2 + self.n_d * self.n_r + self.n_r * (self.n_r - 1) // 2


def make_config(name: str, scale: float = 1.0, seed_offset: int = 0) -> Workload:
    """seed_offset shifts every seed: another realisation of the same configuration."""
    spec = CONFIGS[name]
    n_d = max(2, int(round(spec["n_d"] * scale)))
    n_r = max(2, int(round(spec["n_r"] * scale)))
    sd, sr = (s + seed_offset for s in spec["seeds"])
    cl = spec["cluster"]
    if cl is None:
        ra_d, dec_d = uniform_patch(n_d, spec["ra"], spec["dec"], sd)
    else:
        n_par = max(1, int(round(cl["n_parents"] * scale)))
        if cl["children"] == "fixed":
            per = spec["n_d"] // cl["n_parents"]
            n_d = n_par * per
        ra_d, dec_d = neyman_scott(n_d, n_par, cl["sigma_arcmin"], spec["ra"], spec["dec"], sd,
                                   children=cl["children"], wrap_ra=cl.get("wrap_ra", False))
    ra_r, dec_r = uniform_patch(n_r, spec["ra"], spec["dec"], sr)
    w_d = w_r = None
    if spec["weights"] is not None:
        w_d = lognormal_weights(n_d, spec["weights"][0] + seed_offset)
        w_r = lognormal_weights(n_r, spec["weights"][1] + seed_offset)
    tmin, tmax, nb = spec["bins"]
    theta = log_theta_edges_deg(tmin, tmax, nb)
    return Workload(name=name, scale=scale, ra_d=ra_d, dec_d=dec_d, ra_r=ra_r, dec_r=dec_r,
                    theta_edges_deg=theta, cos_edges=cos_edges_from_theta_deg(theta), w_d=w_d, w_r=w_r,
                    meta=dict(spec=name, ra=spec["ra"], dec=spec["dec"], cluster=cl))
