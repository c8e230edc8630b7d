"""Pins for oracle/fftmodel.py (FFT slope model, Eq.41-46).

The oracle evaluates the continuous integrals of Eq.43 / Eq.46 in PHYSICAL space (edge-averaged structure function).  It is
pinned by an independent route, the Fourier integrals as printed, summed over frequency grids that are refined until they
converge (tests/fourier_sum.py); by adaptive quadrature of Eq.43 (scipy); by its symmetries; by the link to the already pinned
stencil models at large separation; by the convergence of its own quadrature; and end to end (signs).
"""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import covariance as cov
from oracle import fftmodel as fm
from oracle import vonkarman as vk

import fourier_sum as fs

R0, L0, W = 0.15, 6.0, 0.5          # a short outer scale keeps the Riemann grids (df = 1/64 per m and finer) fine against 1/L0

_D = np.array([[0.0, 0.0], [0.5, 0.0], [0.0, 0.5], [0.5, 0.5], [0.25, 0.1], [1.0, -0.5], [2.3, 1.7], [-2.9, 0.4]])


def test_fourier_integrals_as_printed_converge_to_the_physical_space_oracle():
    """Eq.43 / Eq.46 as Riemann sums: truncated at |f| < 2/w (pixel w/4, the library builder's grid) they are within 0.5 % of the
    slope variance of the oracle, and the error falls with the cut-off (|f| < 8/w: below 1e-4): the oracle IS the integral the
    paper prints, with the sign and 2 pi / gamma factors of reading G29."""
    var = fm.cov_slope_slope(np.zeros((1, 2)), 0, 0, W, 1 / W, R0, L0)[0]
    for a, b in ((0, 0), (1, 1), (0, 1), (1, 0)):
        got = fm.cov_slope_slope(_D, a, b, W, 1 / W, R0, L0)
        e_coarse = np.abs(fs.cov_slope_slope(_D, a, b, W, 1 / W, R0, L0, 512, 4) - got).max() / var
        e_fine = np.abs(fs.cov_slope_slope(_D, a, b, W, 1 / W, R0, L0, 2048, 16) - got).max() / var
        assert e_coarse < 5e-3 and e_fine < 1e-4 and e_fine < 0.2 * e_coarse + 1e-6, (a, b, e_coarse, e_fine)
    for b in (0, 1):
        got = fm.cov_phase_slope(_D, b, W, 1 / W, R0, L0)
        sc = np.abs(got).max()
        e_coarse = np.abs(fs.cov_phase_slope(_D, b, W, 1 / W, R0, L0, 512, 4) - got).max() / sc
        e_fine = np.abs(fs.cov_phase_slope(_D, b, W, 1 / W, R0, L0, 2048, 16) - got).max() / sc
        assert e_coarse < 5e-3 and e_fine < 1e-4, (b, e_coarse, e_fine)


def _quad_ss(D, a, b, w, r0, L0, fmax=60.0):
    def g(fy, fx):
        fa, fb = (fx, fy)[a], (fx, fy)[b]
        H = np.sinc(w * fx) * np.sinc(w * fy)
        return (2 * math.pi) ** 2 * fa * fb * vk.psd(math.hypot(fx, fy), r0, L0) * H * H * math.cos(2 * math.pi * (fx * D[0] + fy * D[1]))
    v, _ = integrate.dblquad(g, -fmax, fmax, -fmax, fmax, epsabs=1e-5, epsrel=1e-5)
    return v


@pytest.mark.slow
def test_variance_against_adaptive_quadrature_of_eq43():
    got0 = fm.cov_slope_slope(np.zeros((1, 2)), 0, 0, W, 1.0 / W, R0, L0)[0]
    want0 = _quad_ss((0.0, 0.0), 0, 0, W, R0, L0)
    assert abs(got0 / want0 - 1) < 2e-3, (got0, want0)           # (the quadrature is cut at |f| < 60 / m = 30 / w)


def test_quadrature_of_the_oracle_has_converged():
    base = (fm.cov_slope_slope(_D, 0, 0, W, 1 / W, R0, L0), fm.cov_slope_slope(_D, 0, 1, W, 1 / W, R0, L0), fm.cov_phase_slope(_D, 0, W, 1 / W, R0, L0))
    n1, n2 = fm.N_NODES_1D, fm.N_NODES_2D
    try:
        fm.N_NODES_1D, fm.N_NODES_2D = 3 * n1, 3 * n2
        fine = (fm.cov_slope_slope(_D, 0, 0, W, 1 / W, R0, L0), fm.cov_slope_slope(_D, 0, 1, W, 1 / W, R0, L0), fm.cov_phase_slope(_D, 0, W, 1 / W, R0, L0))
    finally:
        fm.N_NODES_1D, fm.N_NODES_2D = n1, n2
    var = base[0][0]
    for x, y in zip(base, fine):
        assert np.abs(x - y).max() < 1e-7 * var


def test_closed_form_special_cases():
    """Same-axis covariance far across the slope axis (|Dy| >> w) tends to the two-point Hudgin form (edge averaging no longer
    matters), and the x-slope of a subaperture is uncorrelated with its own y-slope and with the phase at its centre."""
    D = np.array([[0.7, 40.0 * W]])
    h = cov.cov_slope_slope(D, 0, 0, W, 1 / W, R0, 25.0, "hudgin")[0]
    f = fm.cov_slope_slope(D, 0, 0, W, 1 / W, R0, 25.0)[0]
    assert abs(f - h) < 2e-3 * abs(h), (f, h)
    z = np.zeros((1, 2))
    v = fm.cov_slope_slope(z, 0, 0, W, 1 / W, R0, L0)[0]
    assert abs(fm.cov_slope_slope(z, 0, 1, W, 1 / W, R0, L0)[0]) < 1e-12 * v
    assert abs(fm.cov_phase_slope(z, 0, W, 1 / W, R0, L0)[0]) < 1e-12 * v


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
    assert abs(fm.cov_phase_slope(np.zeros((1, 2)), 1, W, 1 / W, R0, L0)[0]) < 1e-12 * xx.max()        # Sigma_phi-s(0) = 0
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
