"""Pupil geometry of one n x n Shack-Hartmann WFS (oracle).  Test infrastructure only.

Fig.2 and L132: n x n subapertures, (n+1) x (n+1) phase points on
the subaperture corners; vignetted subapertures and their phase points are dropped
(L301-305).  Readings (G12): a subaperture is valid iff its centre lies
inside the pupil (and outside the central obstruction); a phase point is valid iff
it is a corner of at least one valid subaperture.  Grids are row-major: index
q = iy*n + ix at x = (ix-(n-1)/2) d, y = (iy-(n-1)/2) d; phase point p = iy*(n+1)+ix
at ((ix,iy) - n/2) d.
"""
import math

import numpy as np

ARCSEC = math.pi / (180.0 * 3600.0)


def subap_centres(n: int, d: float):
    """(n*n, 2) centre coordinates [m] of the full square grid."""
    c = (np.arange(n) - (n - 1) / 2.0) * d
    X, Y = np.meshgrid(c, c, indexing="xy")       # row = iy, column = ix
    return np.stack([X.ravel(), Y.ravel()], axis=1)


def phase_points(n: int, d: float):
    """((n+1)^2, 2) corner coordinates [m]."""
    c = (np.arange(n + 1) - n / 2.0) * d
    X, Y = np.meshgrid(c, c, indexing="xy")
    return np.stack([X.ravel(), Y.ravel()], axis=1)


def subap_mask(n: int, D: float, obstruction: float = 0.0):
    """Boolean (n, n): centre within the pupil.  Integer arithmetic on the outer edge:
    |r_q| <= D/2  <=>  (2ix-n+1)^2 + (2iy-n+1)^2 <= n^2   (d = D/n)."""
    k = 2 * np.arange(n) - (n - 1)
    r2 = k[None, :] ** 2 + k[:, None] ** 2
    m = r2 <= n * n
    if obstruction > 0.0:
        m &= r2 >= (obstruction * n) ** 2
    return m


def phase_mask(smask):
    """Boolean (n+1, n+1): corner of at least one valid subaperture."""
    n = smask.shape[0]
    pm = np.zeros((n + 1, n + 1), dtype=bool)
    pm[:-1, :-1] |= smask
    pm[:-1, 1:] |= smask
    pm[1:, :-1] |= smask
    pm[1:, 1:] |= smask
    return pm


def cone_factor(h_k: float, h_gs: float) -> float:
    """gamma_k = (h_gs - h_k)/h_gs (L158); 1 for an NGS."""
    if math.isinf(h_gs):
        return 1.0
    return (h_gs - h_k) / h_gs


def n_prime(n: int, gamma_min: float) -> int:
    """Common size n' of the resampled phase grid (L179, L295; reading G19): the smallest
    integer >= n/gamma_min + 1 with the parity of n+1, so that the ground-layer grid
    coincides with the original phase points."""
    v = n / gamma_min + 1.0
    m = int(math.ceil(v - 1e-9))
    if (m - (n + 1)) % 2 != 0:
        m += 1
    return m
