"""Seeded synthetic sky catalogues: (RA, Dec) in degrees as float64, weights as float32.

Every generator takes a seed, builds numpy.random.default_rng(seed) (PCG64) and
draws in a fixed, documented order, so a (generator, arguments, seed) triple names
one catalogue bit for bit.  No unit vectors or separations are computed here.
"""
from __future__ import annotations

import numpy as np

_DEG = np.pi / 180.0


def _area_uniform(rng, n, ra0, ra1, dec0, dec1):
    """RA ~ U[ra0, ra1), sin(Dec) ~ U[sin dec0, sin dec1).  Draw order: RA, then sin Dec."""
    ra = rng.uniform(ra0, ra1, size=n)
    s = rng.uniform(np.sin(dec0 * _DEG), np.sin(dec1 * _DEG), size=n)
    dec = np.arcsin(np.clip(s, -1.0, 1.0)) / _DEG
    return ra, dec


def uniform_patch(n: int, ra_range, dec_range, seed: int):
    """Area-uniform ('flat'; uniform in sin Dec per BASELINE.json) points on a
    RA/Dec rectangle.  Returns (ra_deg, dec_deg)."""
    rng = np.random.default_rng(seed)
    return _area_uniform(rng, int(n), ra_range[0], ra_range[1], dec_range[0], dec_range[1])


def full_sky(n: int, seed: int):
    """Area-uniform on the whole sphere: RA ~ U[0, 360), sin Dec ~ U[-1, 1)."""
    return uniform_patch(n, (0.0, 360.0), (-90.0, 90.0), seed)


def lognormal_weights(n: int, seed: int, mu: float = 0.0, sigma: float = 0.3) -> np.ndarray:
    """float32 weights, lognormal(mu, sigma) (BASELINE.json config 4)."""
    rng = np.random.default_rng(seed)
    return rng.lognormal(mean=mu, sigma=sigma, size=int(n)).astype(np.float32)


def neyman_scott(n: int, n_parents: int, sigma_arcmin: float, ra_range, dec_range, seed: int,
                 children: str = "fixed", wrap_ra: bool = False):
    """Neyman-Scott cluster process on a RA/Dec rectangle.

    Parents are area-uniform.  A child sits at parent + sigma * (g1 / cos(dec_p), g2)
    in (RA, Dec) with g ~ N(0, 1): an isotropic 2-D Gaussian of width sigma on the
    sky.  'Clipped to patch' is read literally: coordinates are clamped into
    [lo, nextafter(hi, lo)]; with wrap_ra the RA is taken modulo 360 instead.

    children = "fixed":   exactly n / n_parents children per parent (n must divide).
    children = "poisson": m_p ~ Poisson(n / n_parents) per parent; the resulting list
                          is then trimmed (random subset) or padded (extra children of
                          random parents) to exactly n points.
    Draw order: parent RA, parent sin Dec, [Poisson counts], g1, g2, [trim/pad draws].
    """
    n = int(n)
    n_parents = int(n_parents)
    rng = np.random.default_rng(seed)
    pra, pdec = _area_uniform(rng, n_parents, ra_range[0], ra_range[1], dec_range[0], dec_range[1])
    if children == "fixed":
        if n % n_parents:
            raise ValueError("fixed children: n must be a multiple of n_parents")
        owner = np.repeat(np.arange(n_parents), n // n_parents)
    elif children == "poisson":
        m = rng.poisson(n / n_parents, size=n_parents)
        owner = np.repeat(np.arange(n_parents), m)
    else:
        raise ValueError("children must be 'fixed' or 'poisson'")
    g1 = rng.standard_normal(owner.size)
    g2 = rng.standard_normal(owner.size)
    sig = sigma_arcmin / 60.0
    ra = pra[owner] + sig * g1 / np.cos(pdec[owner] * _DEG)
    dec = pdec[owner] + sig * g2
    if children == "poisson" and owner.size != n:
        if owner.size > n:
            keep = np.sort(rng.permutation(owner.size)[:n])
            ra, dec = ra[keep], dec[keep]
        else:
            extra = n - owner.size
            own2 = rng.integers(0, n_parents, size=extra)
            h1 = rng.standard_normal(extra)
            h2 = rng.standard_normal(extra)
            ra = np.concatenate([ra, pra[own2] + sig * h1 / np.cos(pdec[own2] * _DEG)])
            dec = np.concatenate([dec, pdec[own2] + sig * h2])
    if wrap_ra:
        ra = np.mod(ra, 360.0)
        ra[ra >= 360.0] = 0.0
    else:
        ra = np.clip(ra, ra_range[0], np.nextafter(ra_range[1], ra_range[0]))
    dec = np.clip(dec, dec_range[0], np.nextafter(dec_range[1], dec_range[0]))
    return ra, dec
