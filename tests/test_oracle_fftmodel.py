"""Pins for oracle/fftmodel.py (FFT slope model, Eq.41-46).

The defining integrals are checked by an independent route (adaptive quadrature of Eq.43 / Eq.46 in scipy), by their
symmetries, by the link to the already pinned stencil models at large separation (both measure the same gradient there),
and by a Monte-Carlo-free consistency: integrating the x-slope covariance along x recovers phase differences.
"""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import covariance as cov
from oracle import fftmodel as fm
from oracle import vonkarman as vk

R0, L0, W = 0.15, 6.0, 0.5          # a short outer scale keeps the Riemann grid (df = 4/(512 * 0.5) = 1/64 per m) fine against 1/L0


def _quad_ss(D, a, b, w, r0, L0, fmax=40.0):
    def g(fy, fx):
        fa, fb = (fx, fy)[a], (fx, fy)[b]
        H = np.sinc(w * fx) * np.sinc(w * fy)
        return (2 * math.pi) ** 2 * fa * fb * vk.psd(math.hypot(fx, fy), r0, L0) * H * H * math.cos(2 * math.pi * (fx * D[0] + fy * D[1]))
    v, _ = integrate.dblquad(g, -fmax, fmax, -fmax, fmax, epsabs=1e-4, epsrel=1e-4)
    return v


def test_variance_and_one_lag_against_adaptive_quadrature():
    got0 = fm.cov_slope_slope(np.zeros((1, 2)), 0, 0, W, 1.0 / W, R0, L0)[0]
    want0 = _quad_ss((0.0, 0.0), 0, 0, W, R0, L0)
    assert abs(got0 / want0 - 1) < 2e-2, (got0, want0)           # grid truncated at |f| < 4/w, quadrature at 40/m
    D = (0.5, 1.0)
    got = fm.cov_slope_slope(np.array([D]), 0, 1, W, 1.0 / W, R0, L0)[0]
    want = _quad_ss(D, 0, 1, W, R0, L0)
    assert abs(got - want) < 2e-2 * abs(want0), (got, want)


def test_symmetries():
    rng = np.random.default_rng(2)
    D = rng.uniform(-3, 3, size=(6, 2))
    xx = fm.cov_slope_slope(D, 0, 0, W, 1 / W, R0, L0)
    assert np.allclose(xx, fm.cov_slope_slope(-D, 0, 0, W, 1 / W, R0, L0), rtol=1e-12)              # even
    assert np.allclose(fm.cov_slope_slope(D, 0, 1, W, 1 / W, R0, L0), fm.cov_slope_slope(D, 1, 0, W, 1 / W, R0, L0), rtol=1e-12)
    assert np.allclose(xx, fm.cov_slope_slope(D[:, ::-1], 1, 1, W, 1 / W, R0, L0), rtol=1e-12)      # x <-> y
    assert abs(fm.cov_slope_slope(np.zeros((1, 2)), 0, 1, W, 1 / W, R0, L0)[0]) < 1e-12 * xx.max()   # Sigma_sxsy(0) = 0
    ps = fm.cov_phase_slope(D, 0, W, 1 / W, R0, L0)
    assert np.allclose(ps, -fm.cov_phase_slope(-D, 0, W, 1 / W, R0, L0), rtol=1e-12)                # odd
    assert abs(fm.cov_phase_slope(np.zeros((1, 2)), 1, W, 1 / W, R0, L0)[0]) < 1e-15                 # Sigma_phi-s(0) = 0
    # cone compression: slopes scale with gamma (normalisation 1/d, arms gamma d)
    g = 0.8
    a1 = fm.cov_slope_slope(g * D, 0, 0, g * W, 1 / W, R0, L0)
    a2 = fm.cov_slope_slope(g * D, 0, 0, g * W, 1 / (g * W), R0, L0)
    assert np.allclose(a1, g * g * a2, rtol=1e-12)


def test_agrees_with_the_stencil_models_at_large_separation():
    """Far from the subaperture every model measures the same gradient: FFT vs Hudgin within a few per cent at |D| >= 6 w,
    and the same sign structure for the phase-slope covariance."""
    D = np.array([[3.0, 0.0], [0.0, 3.5], [3.0, 2.5], [-4.0, 1.0]])
    for a, b in ((0, 0), (1, 1), (0, 1)):
        f = fm.cov_slope_slope(D, a, b, W, 1 / W, R0, L0)
        h = cov.cov_slope_slope(D, a, b, W, 1 / W, R0, L0, "hudgin")
        scale = np.abs(cov.cov_slope_slope(D, 0, 0, W, 1 / W, R0, L0, "hudgin")).max()
        assert np.abs(f - h).max() < 0.05 * scale, (a, b, f, h)
    for b in (0, 1):
        f = fm.cov_phase_slope(D, b, W, 1 / W, R0, L0)
        h = cov.cov_phase_slope(D, b, W, 1 / W, R0, L0, "hudgin")
        assert np.abs(f - h).max() < 0.05 * np.abs(h).max(), (b, f, h)


def test_model_variance_is_below_hudgin_and_dispatch_through_covariance():
    """Averaging the gradient over the subaperture removes power a two-point difference keeps; and covariance.py reaches
    the model through model='fft'."""
    z = np.zeros((1, 2))
    v_fft = cov.cov_slope_slope(z, 0, 0, W, 1 / W, R0, L0, "fft")[0]
    v_hud = cov.cov_slope_slope(z, 0, 0, W, 1 / W, R0, L0, "hudgin")[0]
    assert 0.5 * v_hud < v_fft < v_hud
    assert v_fft == fm.cov_slope_slope(z, 0, 0, W, 1 / W, R0, L0)[0]


def test_end_to_end_with_the_fft_model_reduces_error_and_pins_signs():
    """MMSE reconstruction with the FFT-model covariances on screen-generated (two-point) slopes: the estimate must follow the
    true phase -- this fixes the sign of Eq.46 and the gamma / 2 pi factors at once (a flipped sign gives an error > 1)."""
    from oracle.system import OracleSystem
    from tomo_inputs import get_config, screens
    from tomo_inputs.configs import small_lgs_config
    for cfg in (get_config("cfg1"), small_lgs_config(n=8, n_gs=3, n_layers=2)):
        s = OracleSystem(cfg, model="fft")
        inp = screens.generate(cfg, s.sigma2)
        phi = s.reconstruct(s.solve_direct(inp["slopes"][0].ravel()))
        truth = s.Mphi @ inp["truth"][0, 0]
        assert np.linalg.norm(phi - truth) / np.linalg.norm(truth) < 0.7
        assert np.corrcoef(phi, truth)[0, 1] > 0.75
        assert np.linalg.norm(-phi - truth) / np.linalg.norm(truth) > 1.2
        w = np.linalg.eigvalsh(s.Css)
        assert w.min() > -1e-9 * w.max()                                  # a covariance matrix
