"""Slope-slope and phase-slope covariances from POSITIONS (oracle, fp64).
Test infrastructure only; no Toeplitz indexing anywhere in this file.

Slope models are linear stencils on the phase (App. A of the paper):
  Hudgin-like, Eq.47-48: s_x = c [phi(r + d_x/2) - phi(r - d_x/2)]
  Fried,       Eq.54-55 (L630-640):          s_x = c/2 [phi_a - phi_b - phi_c + phi_d]
with c = lambda/(2 pi d) -> 1/d here (reading G6: slopes in rad/m).  For any such
stencil {(o_m, w_m)} with sum w = 0,
  cov(s_a(r), s_b(r')) = sum_m sum_m' w_m w'_m' C_phi(r' + o'_m' - r - o_m)
                       = -1/2 sum_m sum_m' w_m w'_m' D_phi(|Delta + o'_m' - o_m|),  Delta = r' - r,
  cov(phi(r_p), s_b(r_q)) = -1/2 sum_m' w'_m' D_phi(|r_q + o'_m' - r_p|),
(Eq.49 L598 and the identity at L600); Eq.50-52 and Eq.56-62 are special cases and are
checked against this function in tests/test_oracle_covariance.py.

A third model, the FFT slope model (Eq.41-46: the gradient averaged over the subaperture), is not a stencil; it
lives in fftmodel.py and is reached through the same two functions with model="fft".

Layers (L562, reading G8): D_phi,k = f_k D_phi, covariances add over layers.
Cone effect (L158, reading G7): at layer k a subaperture of an LGS WFS j sits at
gamma_k r_q + h_k alpha_j, its stencil arms are d_k = gamma_k d long, the
normalisation stays 1/d.
"""
import numpy as np

from . import vonkarman as vk
from .geometry import ARCSEC, cone_factor

# stencil = list of ((ox, oy) in units of the local subaperture width, weight)
STENCILS = {
    "hudgin": {
        0: [((+0.5, 0.0), +1.0), ((-0.5, 0.0), -1.0)],
        1: [((0.0, +0.5), +1.0), ((0.0, -0.5), -1.0)],
    },
    "fried": {
        0: [((+0.5, +0.5), +0.5), ((-0.5, +0.5), -0.5), ((-0.5, -0.5), -0.5), ((+0.5, -0.5), +0.5)],
        1: [((+0.5, +0.5), +0.5), ((-0.5, +0.5), +0.5), ((-0.5, -0.5), -0.5), ((+0.5, -0.5), -0.5)],
    },
}


def _merged_pairs(st_a, st_b):
    """Offsets o'_m' - o_m with their summed weights w_m w'_m' (duplicates merged)."""
    acc = {}
    for (oa, wa) in st_a:
        for (ob, wb) in st_b:
            key = (ob[0] - oa[0], ob[1] - oa[1])
            acc[key] = acc.get(key, 0.0) + wa * wb
    return [(k, w) for k, w in acc.items() if w != 0.0]


def cov_slope_slope(delta, a: int, b: int, width: float, c: float, r0: float, L0: float,
                    model: str = "hudgin"):
    """cov(s_a(r), s_b(r + delta)) for one layer of unit Cn2 fraction.

    delta: (..., 2) separation [m] (second minus first); width: local subaperture size d_k;
    c: slope normalisation (1/d)."""
    if model == "fft":           # subaperture-averaged gradient, Eq.41-45 (not a stencil)
        from . import fftmodel
        return fftmodel.cov_slope_slope(delta, a, b, width, c, r0, L0)
    delta = np.asarray(delta, dtype=np.float64)
    out = np.zeros(delta.shape[:-1])
    for (off, w) in _merged_pairs(STENCILS[model][a], STENCILS[model][b]):
        rx = delta[..., 0] + off[0] * width
        ry = delta[..., 1] + off[1] * width
        out += w * vk.structure_function(np.hypot(rx, ry), r0, L0)
    return -0.5 * c * c * out


def cov_phase_slope(delta, b: int, width: float, c: float, r0: float, L0: float,
                    model: str = "hudgin"):
    """cov(phi(r_p), s_b(r_p + delta)) for one layer of unit Cn2 fraction (delta = r_q - r_p)."""
    if model == "fft":           # Eq.46
        from . import fftmodel
        return fftmodel.cov_phase_slope(delta, b, width, c, r0, L0)
    delta = np.asarray(delta, dtype=np.float64)
    out = np.zeros(delta.shape[:-1])
    for (off, w) in STENCILS[model][b]:
        rx = delta[..., 0] + off[0] * width
        ry = delta[..., 1] + off[1] * width
        out += w * vk.structure_function(np.hypot(rx, ry), r0, L0)
    return -0.5 * c * out


def dense_css(centres_valid, d, wfs_dirs, wfs_hgs, h, frac, r0, L0, model="hudgin"):
    """W_s Sigma_ss W_s^T (Eq.14 L138 / G9, Eq.34) from positions.

    centres_valid: (n_vs, 2) pupil-plane subaperture centres; wfs_dirs: (N, 2) arcsec.
    Ordering of the result: [wfs][component x,y][valid subaperture] (L56, Eq.29)."""
    nv = centres_valid.shape[0]
    N = len(wfs_dirs)
    c = 1.0 / d
    out = np.zeros((N, 2, nv, N, 2, nv))
    for k, (hk, fk) in enumerate(zip(h, frac)):
        for i in range(N):
            gi = cone_factor(hk, wfs_hgs[i])
            pos_i = gi * centres_valid + hk * np.asarray(wfs_dirs[i]) * ARCSEC
            for j in range(i, N):
                gj = cone_factor(hk, wfs_hgs[j])
                if abs(gi - gj) > 1e-15:
                    raise ValueError("mixed guide-star altitudes: not a 2RBT system (L158)")
                pos_j = gj * centres_valid + hk * np.asarray(wfs_dirs[j]) * ARCSEC
                delta = pos_j[None, :, :] - pos_i[:, None, :]
                for a in range(2):
                    for b in range(2):
                        blk = fk * cov_slope_slope(delta, a, b, gi * d, c, r0, L0, model)
                        out[i, a, :, j, b, :] += blk
                        if j != i:
                            out[j, b, :, i, a, :] += blk.T
    return out.reshape(N * 2 * nv, N * 2 * nv)


def dense_cos_direct(phase_pts, centres_valid, d, wfs_dirs, wfs_hgs, beta, h, frac, r0, L0,
                     model="hudgin"):
    """Sigma_{phi_beta s} (Eq.15) from positions, no resampling: target at infinity,
    phase point at r_p + h_k beta, slope of WFS j at gamma_k r_q + h_k alpha_j."""
    npts = phase_pts.shape[0]
    nv = centres_valid.shape[0]
    N = len(wfs_dirs)
    c = 1.0 / d
    out = np.zeros((npts, N, 2, nv))
    for hk, fk in zip(h, frac):
        pp = phase_pts + hk * np.asarray(beta) * ARCSEC
        for j in range(N):
            g = cone_factor(hk, wfs_hgs[j])
            pos_j = g * centres_valid + hk * np.asarray(wfs_dirs[j]) * ARCSEC
            delta = pos_j[None, :, :] - pp[:, None, :]
            for b in range(2):
                out[:, j, b, :] += fk * cov_phase_slope(delta, b, g * d, c, r0, L0, model)
    return out.reshape(npts, N * 2 * nv)


def bilinear_matrix(phase_pts, d_k: float, n_p: int):
    """I'_k of Eq.16 (L189): bilinear weights of the original phase points on the n' x n'
    grid of spacing d_k centred on the target footprint (reading G18); 4 non-zeros per row."""
    npts = phase_pts.shape[0]
    M = np.zeros((npts, n_p * n_p))
    t = phase_pts / d_k + (n_p - 1) / 2.0
    for p in range(npts):
        tx, ty = t[p]
        ix = min(max(int(np.floor(tx + 1e-12)), 0), n_p - 2)
        iy = min(max(int(np.floor(ty + 1e-12)), 0), n_p - 2)
        wx, wy = tx - ix, ty - iy
        if not (-1e-9 <= wx <= 1 + 1e-9 and -1e-9 <= wy <= 1 + 1e-9):
            raise ValueError("phase point outside the resampled grid")
        M[p, iy * n_p + ix] += (1 - wx) * (1 - wy)
        M[p, iy * n_p + ix + 1] += wx * (1 - wy)
        M[p, (iy + 1) * n_p + ix] += (1 - wx) * wy
        M[p, (iy + 1) * n_p + ix + 1] += wx * wy
    return M


def dense_cos_interpolated(phase_pts, centres_valid, d, wfs_dirs, h_gs, beta, h, frac, r0, L0,
                           n_p: int, model="hudgin", return_layers=False):
    """The paper's LGS form Eq.17 (L195): Sigma_{phi s} = sum_k I'_k Xi'_k, with Xi'_k the
    covariance between the slopes and a phase vector on an n' x n' grid of spacing
    d_k = gamma_k d (L179-193), grid point u_p' = (p' - (n'-1)/2) d_k + h_k beta."""
    npts = phase_pts.shape[0]
    nv = centres_valid.shape[0]
    N = len(wfs_dirs)
    c = 1.0 / d
    g1 = (np.arange(n_p) - (n_p - 1) / 2.0)
    GX, GY = np.meshgrid(g1, g1, indexing="xy")
    grid_unit = np.stack([GX.ravel(), GY.ravel()], axis=1)
    out = np.zeros((npts, N * 2 * nv))
    layers = []
    for hk, fk in zip(h, frac):
        g = cone_factor(hk, h_gs)
        dk = g * d
        u = grid_unit * dk + hk * np.asarray(beta) * ARCSEC
        xi = np.zeros((n_p * n_p, N, 2, nv))
        for j in range(N):
            pos_j = g * centres_valid + hk * np.asarray(wfs_dirs[j]) * ARCSEC
            delta = pos_j[None, :, :] - u[:, None, :]
            for b in range(2):
                xi[:, j, b, :] = fk * cov_phase_slope(delta, b, dk, c, r0, L0, model)
        xi = xi.reshape(n_p * n_p, N * 2 * nv)
        Ik = bilinear_matrix(phase_pts, dk, n_p)
        out += Ik @ xi
        if return_layers:
            layers.append((Ik, xi))
    return (out, layers) if return_layers else out
