"""Eq.43 / Eq.46 written out as a Riemann sum over a frequency grid: the discretisation an FFT of edge
n_grid with pixel w / m_over implements (f = p df, p in {-(n_grid/2 - 1), .., n_grid/2 - 1}^2, df = m_over / (n_grid w), the
unpaired Nyquist sample left out).  Test helper, used two ways: on the BUILDER's grid to check the builder's FFT machinery, and
on finer / longer grids as an independent route to the continuous integral that oracle/fftmodel.py evaluates in physical space."""
import math

import numpy as np

from oracle import vonkarman as vk


def _freqs(width, n_grid, m_over):
    df = m_over / (n_grid * width)
    return np.arange(-(n_grid // 2 - 1), n_grid // 2) * df, df


def _factorised_sum(Wc, f, dx, dy, kind):
    ux, ix = np.unique(dx, return_inverse=True)
    uy, iy = np.unique(dy, return_inverse=True)
    M = np.exp(2j * math.pi * np.outer(f, uy)).T @ (Wc @ np.exp(2j * math.pi * np.outer(f, ux)))
    return (M.real if kind == "cos" else M.imag)[iy, ix]


def cov_slope_slope(delta, a, b, width, c, r0, L0, n_grid=512, m_over=4):
    delta = np.asarray(delta, dtype=np.float64)
    f, df = _freqs(width, n_grid, m_over)
    FX, FY = np.meshgrid(f, f, indexing="xy")
    H = np.sinc(width * FX) * np.sinc(width * FY)
    gam = width * c
    W = (gam * gam) * (2 * math.pi) ** 2 * (FX, FY)[a] * (FX, FY)[b] * vk.psd(np.hypot(FX, FY), r0, L0) * H * H * df * df
    return _factorised_sum(W, f, delta[..., 0].ravel(), delta[..., 1].ravel(), "cos").reshape(delta.shape[:-1])


def cov_phase_slope(delta, b, width, c, r0, L0, n_grid=512, m_over=4):
    delta = np.asarray(delta, dtype=np.float64)
    f, df = _freqs(width, n_grid, m_over)
    FX, FY = np.meshgrid(f, f, indexing="xy")
    H = np.sinc(width * FX) * np.sinc(width * FY)
    W = -(width * c) * 2 * math.pi * (FX, FY)[b] * vk.psd(np.hypot(FX, FY), r0, L0) * H * df * df
    return _factorised_sum(W, f, delta[..., 0].ravel(), delta[..., 1].ravel(), "sin").reshape(delta.shape[:-1])
