"""FFT slope model (App. A.A of the paper, Eq.41-46) (oracle, fp64).  Test infrastructure only.

The SH-WFS slope is the phase gradient AVERAGED over the subaperture (Eq.41); its covariances are Fourier
integrals of the von Karman spectrum Phi_phi (Eq.45, constant 0.0229: reading G3) filtered by the subaperture
    H(f) = sinc(w f_x) sinc(w f_y)                                                            (Eq.44)
In this repository's slope unit (rad/m, reading G6: the paper's lambda/2pi factor dropped) and with the cone
compression gamma = w/d of an LGS layer (a pupil-plane gradient is gamma times the layer-plane gradient, L158):
    cov(s_a(r), s_b(r + D))   = gamma^2 int (2 pi)^2 f_a f_b Phi(f) H(f)^2 cos(2 pi f.D) d^2f    (Eq.43)
    cov(phi(r_p), s_b(r_p+D)) = -gamma  int  2 pi f_b      Phi(f) H(f)   sin(2 pi f.D) d^2f      (Eq.46)
(the guide-star shift h_k d_alpha of Eq.43's exponential is part of D here, as everywhere in oracle/).

"In actual computation, the FFT covariance model is computed by the FFT, and its actual accuracy depends on the
sampling" (L572).  Reading G29: the integral is the Riemann sum over the frequency grid an FFT of edge
n_grid with pixel w / m_over has,
    f = p df,  p in {-(n_grid/2 - 1), .., n_grid/2 - 1}^2 (the unpaired Nyquist sample is left out),  df = m_over / (n_grid w),
weights df^2.  This file evaluates that sum DIRECTLY at arbitrary separations (no FFT, no lag lattice): the sum factorises
over the distinct x- and y-separations present in the request.
"""
import math

import numpy as np

from . import vonkarman as vk

N_GRID = 512          # defaults of the reading; the library's builder takes the same two numbers
M_OVER = 4


def _freqs(width: float, n_grid: int, m_over: int):
    df = m_over / (n_grid * width)
    p = np.arange(-(n_grid // 2 - 1), n_grid // 2)
    return p * df, df


def _factorised_sum(Wc, f, dx, dy, kind: str):
    """sum_{fx,fy} Wc[fy, fx] * trig(2 pi (fx dx + fy dy)) for every requested (dx, dy); trig = cos or sin."""
    ux, ix = np.unique(dx, return_inverse=True)
    uy, iy = np.unique(dy, return_inverse=True)
    Ex = np.exp(2j * math.pi * np.outer(f, ux))            # [fx][ux]
    Ey = np.exp(2j * math.pi * np.outer(f, uy))            # [fy][uy]
    M = Ey.T @ (Wc @ Ex)                                    # [uy][ux] = sum W e^{2 pi i (fx dx + fy dy)}
    tab = M.real if kind == "cos" else M.imag
    return tab[iy, ix]


def cov_slope_slope(delta, a: int, b: int, width: float, c: float, r0: float, L0: float,
                    n_grid: int = N_GRID, m_over: int = M_OVER):
    delta = np.asarray(delta, dtype=np.float64)
    f, df = _freqs(width, n_grid, m_over)
    FX, FY = np.meshgrid(f, f, indexing="xy")
    H = np.sinc(width * FX) * np.sinc(width * FY)
    fa = FX if a == 0 else FY
    fb = FX if b == 0 else FY
    gam = width * c
    W = (gam * gam) * (2 * math.pi) ** 2 * fa * fb * vk.psd(np.hypot(FX, FY), r0, L0) * H * H * df * df
    out = _factorised_sum(W, f, delta[..., 0].ravel(), delta[..., 1].ravel(), "cos")
    return out.reshape(delta.shape[:-1])


def cov_phase_slope(delta, b: int, width: float, c: float, r0: float, L0: float,
                    n_grid: int = N_GRID, m_over: int = M_OVER):
    delta = np.asarray(delta, dtype=np.float64)
    f, df = _freqs(width, n_grid, m_over)
    FX, FY = np.meshgrid(f, f, indexing="xy")
    H = np.sinc(width * FX) * np.sinc(width * FY)
    fb = FX if b == 0 else FY
    gam = width * c
    W = -gam * 2 * math.pi * fb * vk.psd(np.hypot(FX, FY), r0, L0) * H * df * df
    out = _factorised_sum(W, f, delta[..., 0].ravel(), delta[..., 1].ravel(), "sin")
    return out.reshape(delta.shape[:-1])
