"""Low-order (tip/tilt) NGS path (oracle, fp64).  Test infrastructure only.

The paper gives no algorithm for the low-order NGS sensors ("we focus only on the high-order correction", PAPER.md
L321, L412; Table 2 L439-449 lists them).  Reading G30 of DESIGN.md: each low-order sensor m at direction beta_m
delivers g_m = (mean valid x-slope, mean valid y-slope) of the full aperture plus white noise of variance sigma2_lo; the
wanted quantity per target t is tau_t = the same aperture-mean slope pair in the target direction; the estimator is the
MMSE one of Eq.5 (L68) written for these small vectors,

    R_lo = C_tau,g (C_gg + sigma2_lo I)^-1          [2T x 2 n_lo],

and the estimated tilt is added back to the (tip/tilt-free, Eq.35) high-order wavefront as tau_x x_p + tau_y y_p over
the valid phase points (slopes are in rad/m, reading G6, so a mean slope IS the tilt coefficient).

Everything here comes from POSITIONS: the covariance of two aperture means is the mean over all pairs of valid
subapertures of the position-based slope covariance of covariance.py (no lag tables, no mask autocorrelation).
"""
import numpy as np

from .covariance import cov_slope_slope
from .geometry import ARCSEC


def mean_slope_covariance(centres_valid, d, dirs, h, frac, r0, L0, model="hudgin"):
    """Covariance of the aperture-mean slope pairs of NGS directions `dirs` ((M, 2) arcsec): (2M, 2M), order [m][x,y]."""
    dirs = np.asarray(dirs, dtype=np.float64).reshape(-1, 2)
    M = dirs.shape[0]
    out = np.zeros((M, 2, M, 2))
    for hk, fk in zip(h, frac):
        for i in range(M):
            pos_i = centres_valid + hk * dirs[i] * ARCSEC
            for j in range(M):
                pos_j = centres_valid + hk * dirs[j] * ARCSEC
                delta = pos_j[None, :, :] - pos_i[:, None, :]
                for a in range(2):
                    for b in range(2):
                        out[i, a, j, b] += fk * cov_slope_slope(delta, a, b, d, 1.0 / d, r0, L0, model).mean()
    return out.reshape(2 * M, 2 * M)


def lo_estimator(centres_valid, d, lo_dirs, targets, h, frac, r0, L0, sigma2_lo, model="hudgin"):
    """R_lo = C_tau,g (C_gg + sigma2_lo I)^-1, shape (2T, 2 n_lo)."""
    lo_dirs = np.asarray(lo_dirs, dtype=np.float64).reshape(-1, 2)
    targets = np.asarray(targets, dtype=np.float64).reshape(-1, 2)
    n_g = 2 * lo_dirs.shape[0]
    Cm = mean_slope_covariance(centres_valid, d, np.concatenate([lo_dirs, targets]), h, frac, r0, L0, model)
    Cgg = Cm[:n_g, :n_g] + sigma2_lo * np.eye(n_g)
    Ctg = Cm[n_g:, :n_g]
    return np.linalg.solve(Cgg, Ctg.T).T


def lo_addback(R_lo, g, phase_pts_valid):
    """tau = R_lo g; returns (T, n_vphi): tau_x x_p + tau_y y_p.  g: (n_lo, 2) mean slopes [rad/m]."""
    tau = (R_lo @ np.asarray(g, dtype=np.float64).reshape(-1)).reshape(-1, 2)
    return tau[:, 0:1] * phase_pts_valid[None, :, 0] + tau[:, 1:2] * phase_pts_valid[None, :, 1]
