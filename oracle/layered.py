"""Layered-phase (MCAO) variant of the spatio-angular reconstructor (oracle, fp64).  Test infrastructure only.

PAPER.md L199 (S2.D, last paragraph): "If we extend the new phase grid to cover the range of the layered phase and
remove the bi-linear interpolation by I'_k, the layered phase at each altitude can be estimated by the spatioangular
reconstructor with the 2RBT formulation. This needs more computation than the directional phase reconstructor, but can
be applicable to MCAO systems."; L516 (S6): "... usable also in MCAO with the caveat that the calculations depend
explicitly on number of estimated layers."

What that defines.  The MMSE estimate (Eq.5, Eq.12-13) of the phase phi_k of layer k ALONE, at the points u
of a square grid laid over the layer's meta-pupil, from the slopes of all WFSs:
    phi_hat_k = Sigma_{phi_k s} W_s^T M_s^T zeta,      (Sigma_ss + Sigma_eta) zeta = s   (same system, same zeta)
    Sigma_{phi_k s}[u, (j, b, q)] = f_k cov( phi(u), s_b at gamma_k r_q + h_k alpha_j )          (layers independent, L90)
i.e. the Xi'_{q,k} of L193 on a LARGER grid, not multiplied by I'_k and not summed over k (Eq.17 L195 is the sum).

Readings (G31):
  - grid of layer k: n_m x n_m points u_m = (m - (n_m - 1)/2) d_k, spacing d_k = gamma_k d (L179-181, the spacing that
    keeps Xi'_k 2RBT against the subaperture grid), centred on the optical axis (the new grid of Eq.16 with beta = 0);
  - one common n_m for all layers (as n' is common, L295 / G19): the smallest integer with the parity of n + 1 that is
    >= max_k (D + 2 h_k theta)/d_k + 1, theta = the field radius the layers must cover; theta = 0 gives back n';
  - the whole square grid is returned: no pupil mask W_phi and no modal removal M_phi in layer space (the paper defines
    both on the pupil-plane phase only, Eq.35).
"""
import math

import numpy as np

from .covariance import cov_phase_slope
from .geometry import ARCSEC, cone_factor


def n_meta(n: int, d: float, h, h_gs: float, fov_radius_arcsec: float) -> int:
    """Common edge n_m of the layer grids (reading G31)."""
    v = max((n * d + 2.0 * hk * fov_radius_arcsec * ARCSEC) / (cone_factor(hk, h_gs) * d) + 1.0 for hk in h)
    m = int(math.ceil(v - 1e-9))
    if (m - (n + 1)) % 2 != 0:
        m += 1
    return m


def layer_grid(n_m: int, d_k: float):
    """(n_m^2, 2) grid points [m] in the layer plane, row-major (row = y)."""
    g1 = (np.arange(n_m) - (n_m - 1) / 2.0) * d_k
    GX, GY = np.meshgrid(g1, g1, indexing="xy")
    return np.stack([GX.ravel(), GY.ravel()], axis=1)


def dense_layer_cov(k: int, n_m: int, centres_valid, d, wfs_dirs, h_gs, h, frac, r0, L0, model="hudgin"):
    """Sigma_{phi_k s}: (n_m^2, N*2*nv), columns ordered [wfs][component][valid subaperture] (Eq.29), built from
    POSITIONS: layer point u against the slope sample point gamma_k r_q + h_k alpha_j of width gamma_k d."""
    hk, fk = h[k], frac[k]
    g = cone_factor(hk, h_gs)
    u = layer_grid(n_m, g * d)
    N, nv = len(wfs_dirs), centres_valid.shape[0]
    out = np.zeros((n_m * n_m, N, 2, nv))
    for j in range(N):
        pos_j = g * centres_valid + hk * np.asarray(wfs_dirs[j]) * ARCSEC
        delta = pos_j[None, :, :] - u[:, None, :]
        for b in range(2):
            out[:, j, b, :] = fk * cov_phase_slope(delta, b, g * d, 1.0 / d, r0, L0, model)
    return out.reshape(n_m * n_m, N * 2 * nv)


def layered_estimate(z, n_m, centres_valid, d, wfs_dirs, h_gs, h, frac, r0, L0, model="hudgin"):
    """phi_hat[k] = Sigma_{phi_k s} z for every layer: (K, n_m, n_m).  z = W_s^T M_s^T zeta (already projected)."""
    return np.stack([(dense_layer_cov(k, n_m, centres_valid, d, wfs_dirs, h_gs, h, frac, r0, L0, model) @ z)
                     .reshape(n_m, n_m) for k in range(len(h))])


def ray_trace(layers, pts, d, h_gs, h, beta_arcsec):
    """Pupil-plane phase of a target at infinity in direction beta (Eq.2 L47 with gamma = 1 for the target): sum over the
    layers of the bilinear interpolate of layer k at r + h_k beta.  layers: (K, n_m, n_m) on layer_grid(n_m, gamma_k d)."""
    K, n_m, _ = layers.shape
    out = np.zeros(pts.shape[0])
    for k in range(K):
        dk = cone_factor(h[k], h_gs) * d
        t = (pts + h[k] * np.asarray(beta_arcsec) * ARCSEC) / dk + (n_m - 1) / 2.0
        if t.min() < -1e-9 or t.max() > n_m - 1 + 1e-9:
            raise ValueError("ray leaves the layer grid")
        i0 = np.clip(np.floor(t + 1e-12).astype(int), 0, n_m - 2)
        w = t - i0
        g = layers[k]
        out += ((1 - w[:, 0]) * (1 - w[:, 1]) * g[i0[:, 1], i0[:, 0]] + w[:, 0] * (1 - w[:, 1]) * g[i0[:, 1], i0[:, 0] + 1]
                + (1 - w[:, 0]) * w[:, 1] * g[i0[:, 1] + 1, i0[:, 0]] + w[:, 0] * w[:, 1] * g[i0[:, 1] + 1, i0[:, 0] + 1])
    return out
