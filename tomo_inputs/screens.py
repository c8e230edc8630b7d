"""Seeded synthetic slopes: von Karman phase screens sampled by a Hudgin-like Shack-Hartmann.

Inputs only -- none of the reconstruction method's arithmetic lives here.  The recipe
 stands in for the paper's OOMAO simulations (PAPER.md L366,
L412-424): per layer one periodic FFT screen with the von Karman spectrum (Eq.45 L559 with
the exact constant 0.02290), r0_k = r0 f_k^{-3/5}; the slope of subaperture q of WFS j is the
difference of the phase at the two edge mid-points (Eq.47-48), ray-traced through
the layers with the LGS cone compression (L158), divided by d; i.i.d. Gaussian noise of a
given variance is added (Eq.2).  The true target phase is kept for sanity checks.
"""
from __future__ import annotations

import math

import numpy as np

from .configs import BASE_SEED, TomoConfig

ARCSEC = math.pi / (180.0 * 3600.0)
_PSD_CONST = 0.022895587


def subap_mask(n: int, obstruction: float = 0.0):
    k = 2 * np.arange(n) - (n - 1)
    r2 = k[None, :] ** 2 + k[:, None] ** 2
    m = r2 <= n * n
    if obstruction > 0:
        m &= r2 >= (obstruction * n) ** 2
    return m


def phase_mask(sm):
    n = sm.shape[0]
    pm = np.zeros((n + 1, n + 1), dtype=bool)
    pm[:-1, :-1] |= sm
    pm[:-1, 1:] |= sm
    pm[1:, :-1] |= sm
    pm[1:, 1:] |= sm
    return pm


def make_screen(npx: int, pixel: float, r0: float, L0: float, rng) -> np.ndarray:
    """One periodic von Karman screen [rad], npx x npx, pixel size [m]."""
    df = 1.0 / (npx * pixel)
    fx = np.fft.fftfreq(npx, d=pixel)
    f2 = fx[None, :] ** 2 + fx[:, None] ** 2
    phi = _PSD_CONST * r0 ** (-5.0 / 3.0) * (f2 + 1.0 / L0 ** 2) ** (-11.0 / 6.0)
    xi = rng.standard_normal((npx, npx)) + 1j * rng.standard_normal((npx, npx))
    return np.real(np.fft.fft2(xi * np.sqrt(phi) * df))


def _bilinear(screen: np.ndarray, pixel: float, xy: np.ndarray) -> np.ndarray:
    """Periodic bilinear sample at xy [m] (origin at the screen centre)."""
    npx = screen.shape[0]
    t = xy / pixel + npx / 2.0
    i0 = np.floor(t).astype(np.int64)
    w = t - i0
    ix0 = i0[:, 0] % npx
    iy0 = i0[:, 1] % npx
    ix1 = (ix0 + 1) % npx
    iy1 = (iy0 + 1) % npx
    wx, wy = w[:, 0], w[:, 1]
    return ((1 - wx) * (1 - wy) * screen[iy0, ix0] + wx * (1 - wy) * screen[iy0, ix1]
            + (1 - wx) * wy * screen[iy1, ix0] + wx * wy * screen[iy1, ix1])


def generate(cfg: TomoConfig, sigma2: float, n_frames: int = 1, seed_offset: int = 0):
    """Returns dict(slopes[n_frames, N, 2, n_vs] fp64, noise-free slopes, truth[n_targets, n_vphi]).

    Frames share the screens and differ in the noise draw and in a rigid shift of the
    screens (frame f is shifted by f * 0.37 m in x: a frozen-flow stand-in), so a batch holds
    distinct but equally distributed slope vectors."""
    n, d = cfg.n, cfg.d
    sm = subap_mask(n, cfg.obstruction)
    pm = phase_mask(sm)
    sidx = np.flatnonzero(sm.ravel())
    pidx = np.flatnonzero(pm.ravel())
    c1 = (np.arange(n) - (n - 1) / 2.0) * d
    cx, cy = np.meshgrid(c1, c1, indexing="xy")
    centres = np.stack([cx.ravel(), cy.ravel()], axis=1)[sidx]
    p1 = (np.arange(n + 1) - n / 2.0) * d
    px, py = np.meshgrid(p1, p1, indexing="xy")
    ppts = np.stack([px.ravel(), py.ravel()], axis=1)[pidx]
    nv = sidx.size
    N = cfg.n_wfs
    pixel = d / 4.0
    base = BASE_SEED + 1000 * cfg.cfg_id + seed_offset
    slopes0 = np.zeros((n_frames, N, 2, nv))
    truth = np.zeros((n_frames, len(cfg.targets), pidx.size))
    ex = np.array([1.0, 0.0])
    ey = np.array([0.0, 1.0])
    for k, (hk, fk) in enumerate(zip(cfg.h, cfg.frac)):
        rng = np.random.default_rng(base + k)
        scr = make_screen(cfg.screen_npx, pixel, cfg.r0 * fk ** (-3.0 / 5.0), cfg.L0, rng)
        for f in range(n_frames):
            shift = np.array([0.37 * f, 0.0])
            for j, w in enumerate(cfg.wfs):
                g = 1.0 if math.isinf(w.h_gs) else (w.h_gs - hk) / w.h_gs
                pos = g * centres + hk * np.array([w.ax, w.ay]) * ARCSEC + shift
                half = 0.5 * g * d
                slopes0[f, j, 0] += (_bilinear(scr, pixel, pos + half * ex)
                                     - _bilinear(scr, pixel, pos - half * ex)) / d
                slopes0[f, j, 1] += (_bilinear(scr, pixel, pos + half * ey)
                                     - _bilinear(scr, pixel, pos - half * ey)) / d
            for t, beta in enumerate(cfg.targets):
                truth[f, t] += _bilinear(scr, pixel, ppts + hk * np.array(beta) * ARCSEC + shift)
    slopes = slopes0.copy()
    for f in range(n_frames):
        rng = np.random.default_rng(base + 500 + f)
        slopes[f] += math.sqrt(sigma2) * rng.standard_normal((N, 2, nv))
    return dict(slopes=slopes, slopes_noiseless=slopes0, truth=truth,
                sub_idx=sidx, phase_idx=pidx, centres=centres, phase_pts=ppts)


def elongated_noise_blocks(cfg: TomoConfig, sigma2: float, elongation: float = 2.0):
    """Synthetic 2 x 2 noise blocks for elongated LGS spots (PAPER.md L331-333 states the structure -- noise that depends on
    the subaperture position relative to the laser launch telescope, plus an x-y cross term -- but no formula).  Recipe: side
    launch from the pupil edge towards guide star i, launch_i = D/2 (cos t_i, sin t_i); a subaperture at r sees the spot
    stretched along e = r - launch_i:  block = sigma2 [I + elongation (|e|/D)^2 e^ e^T].
    Returns (sxx, syy, sxy), each [n_wfs][n_vs], and `with_noise(slopes_noiseless, frame)` drawing noise of that covariance."""
    n, d = cfg.n, cfg.d
    sidx = np.flatnonzero(subap_mask(n, cfg.obstruction).ravel())
    c1 = (np.arange(n) - (n - 1) / 2.0) * d
    cx, cy = np.meshgrid(c1, c1, indexing="xy")
    centres = np.stack([cx.ravel(), cy.ravel()], axis=1)[sidx]
    sxx, syy, sxy = (np.zeros((cfg.n_wfs, sidx.size)) for _ in range(3))
    for i, w in enumerate(cfg.wfs):
        t = math.atan2(w.ay, w.ax)
        e = centres - 0.5 * cfg.D * np.array([math.cos(t), math.sin(t)])
        ln = np.maximum(np.hypot(e[:, 0], e[:, 1]), 1e-12)
        ux, uy = e[:, 0] / ln, e[:, 1] / ln
        extra = sigma2 * elongation * (ln / cfg.D) ** 2
        sxx[i], syy[i], sxy[i] = sigma2 + extra * ux * ux, sigma2 + extra * uy * uy, extra * ux * uy
    return sxx, syy, sxy


def add_block_noise(cfg: TomoConfig, slopes_noiseless: np.ndarray, blocks, seed_offset: int = 0) -> np.ndarray:
    """slopes_noiseless[n_frames, N, 2, n_vs] + zero-mean Gaussian noise with the 2 x 2 covariance blocks (Cholesky factor
    of each block applied to two i.i.d. normals)."""
    sxx, syy, sxy = blocks
    out = np.array(slopes_noiseless, dtype=np.float64, copy=True)
    l11 = np.sqrt(sxx)
    l21 = sxy / l11
    l22 = np.sqrt(np.maximum(syy - l21 * l21, 0.0))
    for f in range(out.shape[0]):
        rng = np.random.default_rng(BASE_SEED + 1000 * cfg.cfg_id + 700 + seed_offset + f)
        z = rng.standard_normal((2,) + sxx.shape)
        out[f, :, 0] += l11 * z[0]
        out[f, :, 1] += l21 * z[0] + l22 * z[1]
    return out


def random_vector(cfg: TomoConfig, length: int, seed_offset: int = 0) -> np.ndarray:
    """A seeded white Gaussian vector (for MVM parity on non-slope-like inputs)."""
    rng = np.random.default_rng(BASE_SEED + 1000 * cfg.cfg_id + 900 + seed_offset)
    return rng.standard_normal(length)
