"""Pins for oracle/covariance.py: the generic stencil evaluation against the formulas the
paper prints (Eq.50-52 L602-613 with reading G4, Eq.56-62), symmetries, limits."""
import numpy as np
import pytest

from oracle import covariance as cov
from oracle import geometry as geo
from oracle import vonkarman as vk
from tomo_inputs import get_config
from tomo_inputs.configs import small_lgs_config

R0, L0 = 0.15, 25.0


def D(v):
    v = np.asarray(v, dtype=float)
    return vk.structure_function(np.hypot(v[..., 0], v[..., 1]), R0, L0)


RNG = np.random.default_rng(7)
DELTAS = np.concatenate([RNG.uniform(-6, 6, size=(40, 2)), np.zeros((1, 2)),
                         np.array([[0.5, 0.0], [0.0, -0.5], [0.25, 0.25]])])


@pytest.mark.parametrize("w", [0.5, 0.37])
def test_hudgin_printed_formulas(w):
    c = 1.0 / 0.5
    dx, dy = np.array([w, 0.0]), np.array([0.0, w])
    d = DELTAS
    xx = 0.5 * c * c * (-2 * D(d) + D(d + dx) + D(d - dx))                                   # Eq.50
    yy = 0.5 * c * c * (-2 * D(d) + D(d + dy) + D(d - dy))                                   # L608 (G5)
    xy = 0.5 * c * c * (D(d + dx / 2 + dy / 2) - D(d - dx / 2 + dy / 2)
                        - D(d + dx / 2 - dy / 2) + D(d - dx / 2 - dy / 2))                  # Eq.51 with G4 (+)
    px = 0.5 * c * (D(d - dx / 2) - D(d + dx / 2))                                           # Eq.52
    py = 0.5 * c * (D(d - dy / 2) - D(d + dy / 2))                                           # L615 (G5)
    assert np.allclose(cov.cov_slope_slope(d, 0, 0, w, c, R0, L0), xx, rtol=0, atol=1e-10)
    assert np.allclose(cov.cov_slope_slope(d, 1, 1, w, c, R0, L0), yy, rtol=0, atol=1e-10)
    assert np.allclose(cov.cov_slope_slope(d, 0, 1, w, c, R0, L0), xy, rtol=0, atol=1e-10)
    assert np.allclose(cov.cov_slope_slope(d, 1, 0, w, c, R0, L0), xy, rtol=0, atol=1e-10)   # L606: sxsy = sysx
    assert np.allclose(cov.cov_phase_slope(d, 0, w, c, R0, L0), px, rtol=0, atol=1e-10)
    assert np.allclose(cov.cov_phase_slope(d, 1, w, c, R0, L0), py, rtol=0, atol=1e-10)


def test_eq51_printed_sign_is_wrong():
    # With the sign as printed (last term negative) an x- and a y-slope of the SAME subaperture
    # would be correlated; symmetry says they are not (reading G4).
    c, w = 2.0, 0.5
    dx, dy = np.array([w, 0.0]), np.array([0.0, w])
    z = np.zeros((1, 2))
    printed = 0.5 * c * c * (D(z + dx / 2 + dy / 2) - D(z - dx / 2 + dy / 2)
                             - D(z + dx / 2 - dy / 2) - D(z - dx / 2 - dy / 2))
    assert abs(printed[0]) > 10.0
    assert abs(cov.cov_slope_slope(z, 0, 1, w, c, R0, L0)[0]) < 1e-12


def test_fried_printed_formulas():
    w = 0.5
    c = 1.0 / w
    dx, dy = np.array([w, 0.0]), np.array([0.0, w])
    d = DELTAS
    F1 = D(d + dx) + D(d - dx)
    F2 = D(d + dy) + D(d - dy)
    F3 = D(d + dx + dy) + D(d - dx - dy)
    F4 = D(d + dx - dy) + D(d - dx + dy)
    k = 0.5 * (c / 2) ** 2
    xx = k * (-4 * D(d) + 2 * F1 - 2 * F2 + F3 + F4)      # Eq.56
    yy = k * (-4 * D(d) - 2 * F1 + 2 * F2 + F3 + F4)      # Eq.57
    xy = k * (F3 - F4)                                    # Eq.58
    F5 = D(d + dx / 2 + dy / 2)
    F6 = D(d - dx / 2 + dy / 2)
    F7 = D(d - dx / 2 - dy / 2)
    F8 = D(d + dx / 2 - dy / 2)
    px = (c / 4) * (-F5 + F6 + F7 - F8)                   # Eq.60
    py = (c / 4) * (-F5 - F6 + F7 + F8)                   # Eq.61
    assert np.allclose(cov.cov_slope_slope(d, 0, 0, w, c, R0, L0, "fried"), xx, atol=1e-10, rtol=0)
    assert np.allclose(cov.cov_slope_slope(d, 1, 1, w, c, R0, L0, "fried"), yy, atol=1e-10, rtol=0)
    assert np.allclose(cov.cov_slope_slope(d, 0, 1, w, c, R0, L0, "fried"), xy, atol=1e-10, rtol=0)
    assert np.allclose(cov.cov_phase_slope(d, 0, w, c, R0, L0, "fried"), px, atol=1e-10, rtol=0)
    assert np.allclose(cov.cov_phase_slope(d, 1, w, c, R0, L0, "fried"), py, atol=1e-10, rtol=0)


def test_zero_lag_values():
    d = 0.5
    z = np.zeros((1, 2))
    v = cov.cov_slope_slope(z, 0, 0, d, 1 / d, R0, L0)[0]
    assert abs(v - float(vk.structure_function(d, R0, L0)) / d ** 2) < 1e-10   # variance = c^2 D(d)
    assert abs(cov.cov_phase_slope(z, 0, d, 1 / d, R0, L0)[0]) < 1e-12
    assert abs(cov.cov_phase_slope(z, 1, d, 1 / d, R0, L0)[0]) < 1e-12


def test_monte_carlo_definition():
    # cov of actual phase differences drawn from the phase covariance C_phi (Cholesky of a small
    # dense phase covariance) reproduces the stencil formula: pins sign and the -1/2 factor.
    d = 0.5
    pts = np.array([[0.25, 0.0], [-0.25, 0.0], [1.3, 0.95], [1.3, 0.45], [0.9, 0.1]])
    R = np.hypot(pts[:, None, 0] - pts[None, :, 0], pts[:, None, 1] - pts[None, :, 1])
    C = vk.phase_covariance(R, R0, L0)
    # exact second moments instead of sampling: s_x(0) = (phi0 - phi1)/d, s_y(r') = (phi2 - phi3)/d
    wx = np.array([1, -1, 0, 0, 0]) / d
    wy = np.array([0, 0, 1, -1, 0]) / d
    exact_xy = wx @ C @ wy
    delta = np.array([[1.3, 0.7]])
    assert abs(cov.cov_slope_slope(delta, 0, 1, d, 1 / d, R0, L0)[0] - exact_xy) < 1e-9
    e4 = np.array([0, 0, 0, 0, 1.0])
    exact_px = e4 @ C @ wx          # cov(phi(p4), s_x at 0): delta = r_q - r_p = -p4
    assert abs(cov.cov_phase_slope(-pts[4:5], 0, d, 1 / d, R0, L0)[0] - exact_px) < 1e-9


def _small_css(cfg):
    n, d = cfg.n, cfg.d
    sm = geo.subap_mask(n, cfg.D)
    cen = geo.subap_centres(n, d)[np.flatnonzero(sm.ravel())]
    dirs = [(w.ax, w.ay) for w in cfg.wfs]
    hgs = [w.h_gs for w in cfg.wfs]
    return cen, cov.dense_css(cen, d, dirs, hgs, cfg.h, cfg.frac, cfg.r0, cfg.L0)


def test_css_symmetric_psd_cfg1():
    cfg = get_config("cfg1")
    cen, C = _small_css(cfg)
    assert C.shape == (208, 208)
    assert np.allclose(C, C.T, atol=1e-9)
    w = np.linalg.eigvalsh(C)
    assert w.min() > 0
    assert abs(C[0, 0] - 122.5555184) < 1e-6      # c^2 D_phi(d), d = 0.5, r0 = 0.15, L0 = 25


def test_single_ground_layer_blocks_identical():
    from dataclasses import replace
    cfg = replace(get_config("cfg1"), h=(0.0,), frac=(1.0,))
    cen, C = _small_css(cfg)
    nv = cen.shape[0]
    B = C.reshape(2, 2 * nv, 2, 2 * nv)
    assert np.allclose(B[0, :, 0, :], B[0, :, 1, :], atol=1e-10)
    assert np.allclose(B[0, :, 0, :], B[1, :, 1, :], atol=1e-10)


def test_lgs_at_infinity_is_ngs():
    from dataclasses import replace
    from tomo_inputs.configs import WFS
    cfg = small_lgs_config(n=6, n_gs=2, n_layers=2, D=3.0)
    far = replace(cfg, wfs=tuple(WFS(w.ax, w.ay, 1e15, w.n_remove) for w in cfg.wfs))
    ngs = replace(cfg, wfs=tuple(WFS(w.ax, w.ay, float("inf"), w.n_remove) for w in cfg.wfs))
    _, Cf = _small_css(far)
    _, Cn = _small_css(ngs)
    assert np.allclose(Cf, Cn, atol=1e-7)
    _, Cl = _small_css(cfg)
    assert not np.allclose(Cl, Cn, atol=1e-3)       # the cone effect matters at 90 km


def test_mixed_altitudes_rejected():
    from dataclasses import replace
    from tomo_inputs.configs import WFS
    cfg = small_lgs_config(n=4, n_gs=2, n_layers=2, D=2.0)
    mixed = replace(cfg, wfs=(cfg.wfs[0], WFS(5.0, 0.0, float("inf"), 0)))
    with pytest.raises(ValueError):
        _small_css(mixed)
