"""Pins of the layered-phase (MCAO) oracle, oracle/layered.py (PAPER.md L199 S2.D, L516 S6; reading G31).

None of these retypes cov_phase_slope: they pin the grid, its centring and ordering, the per-layer split and the cone
geometry against (a) the joint Gaussian model written out sample by sample with the phase COVARIANCE B (not the structure
function), (b) the LTAO covariances of covariance.py, which have their own pins, through ray tracing, (c) the 2RBT product.
"""
from dataclasses import replace

import numpy as np
import pytest

from oracle import covariance as cov
from oracle import geometry as geo
from oracle import layered as lay
from oracle import toeplitz as tz
from oracle import vonkarman as vk
from oracle.system import OracleSystem
from tomo_inputs import get_config
from tomo_inputs.configs import small_lgs_config


def _system(cfg):
    return OracleSystem(cfg, build_cos=False)


def test_n_meta_reduces_to_n_prime_and_grows_with_the_field():
    h = (0.0, 4000.0, 16000.0)
    for n, hgs in [(8, 90e3), (20, 90e3), (74, 90e3), (16, float("inf"))]:
        gmin = min(geo.cone_factor(hk, hgs) for hk in h)
        assert lay.n_meta(n, 0.5, h, hgs, 0.0) == geo.n_prime(n, gmin)            # theta = 0: the LTAO grid (L179)
    # NGS, 16 km, 60 arcsec radius: D + 2 h theta = 8 + 9.308 m over d = 0.5 -> 34.6 + 1 -> 36 -> 37 (parity of n + 1 = 17)
    assert lay.n_meta(16, 0.5, h, float("inf"), 60.0) == 37
    assert lay.n_meta(16, 0.5, h, float("inf"), 30.0) < lay.n_meta(16, 0.5, h, float("inf"), 60.0)
    assert (lay.n_meta(16, 0.5, h, 90e3, 45.0) - 17) % 2 == 0


def test_layer_grid_is_centred_row_major_with_x_fastest():
    u = lay.layer_grid(5, 0.25)
    assert u.shape == (25, 2)
    assert np.allclose(u[0], (-0.5, -0.5)) and np.allclose(u[1], (-0.25, -0.5)) and np.allclose(u[5], (-0.5, -0.25))
    assert np.allclose(u.mean(axis=0), 0.0) and np.allclose(u[12], 0.0)


@pytest.mark.parametrize("lgs", [False, True])
def test_layer_covariance_from_the_joint_gaussian_model_sample_by_sample(lgs):
    """Definition check: lay phase samples on the layer (the grid points and the two end points of every Hudgin slope,
    Eq.47, at gamma_k r_q + h_k alpha_j -+ gamma_k d/2), give them the von Karman COVARIANCE f_k B(|.|), write the
    slopes as the explicit linear map s = sum_k G_k phi_k: then Sigma_{phi_k s} = C_k[grid, ends] G_k^T, and the same
    maps give Sigma_ss = sum_k G_k C_k G_k^T, which must be covariance.dense_css (pinned on its own)."""
    cfg = small_lgs_config(n=4, n_gs=2, n_layers=2) if lgs else replace(get_config("cfg1"), n=4, D=2.0)
    s = _system(cfg)
    c = cfg
    n_m = lay.n_meta(s.n, s.d, c.h, s.h_gs, 20.0)
    css = np.zeros((s.Ns, s.Ns))
    for k, (hk, fk) in enumerate(zip(c.h, c.frac)):
        g = geo.cone_factor(hk, s.h_gs)
        grid = lay.layer_grid(n_m, g * s.d)
        ends, G = [], np.zeros((s.Ns, 2 * s.Ns))
        row = 0
        for j in range(s.N):
            for b in range(2):
                e = np.array([0.5 * g * s.d, 0.0]) if b == 0 else np.array([0.0, 0.5 * g * s.d])
                for q in range(s.nv):
                    pos = g * s.centres[q] + hk * np.asarray(s.dirs[j]) * geo.ARCSEC
                    ends += [pos + e, pos - e]
                    G[row, 2 * row], G[row, 2 * row + 1] = 1.0 / s.d, -1.0 / s.d
                    row += 1
        pts = np.vstack([grid, np.array(ends)])
        Ck = fk * vk.phase_covariance(np.linalg.norm(pts[:, None, :] - pts[None, :, :], axis=-1), c.r0, c.L0)
        ng = grid.shape[0]
        want = Ck[:ng, ng:] @ G.T
        got = lay.dense_layer_cov(k, n_m, s.centres, s.d, s.dirs, s.h_gs, c.h, c.frac, c.r0, c.L0)
        assert np.allclose(got, want, atol=1e-9 * np.abs(want).max())
        css += G @ Ck[ng:, ng:] @ G.T
    ref = cov.dense_css(s.centres, s.d, s.dirs, s.hgs, c.h, c.frac, c.r0, c.L0)
    assert np.allclose(css, ref, atol=1e-9 * np.abs(ref).max())


def test_single_ground_layer_is_the_ltao_covariance_for_any_target():
    """h = 0: the layer IS the pupil, every direction sees the same phase: rows of Sigma_{phi_0 s} at the pupil's phase
    points equal Sigma_{phi_beta s} (Eq.15) whatever beta (verdict r1, item 7 pin i)."""
    cfg = replace(small_lgs_config(n=8, n_gs=3, n_layers=1), h=(0.0,), frac=(1.0,))
    s = _system(cfg)
    n_m = s.n + 3                                              # a grid larger than the pupil; same parity as n + 1
    L = lay.dense_layer_cov(0, n_m, s.centres, s.d, s.dirs, s.h_gs, cfg.h, cfg.frac, cfg.r0, cfg.L0)
    iy, ix = np.divmod(s.ph_idx, s.n + 1)
    sel = (iy + 1) * n_m + (ix + 1)                            # (n_m - (n + 1))/2 = 1 point of margin per side
    assert np.allclose(lay.layer_grid(n_m, s.d)[sel], s.phase_pts)
    for beta in [(0.0, 0.0), (7.0, -4.0)]:
        assert np.allclose(L[sel], s.dense_cos_direct(beta), atol=1e-12)


def test_ray_tracing_the_layers_reproduces_the_ngs_ltao_estimate():
    """NGS system, target direction chosen so that h_k beta is a whole number of grid steps in every layer: the rays hit
    grid points, the bilinear weights are 0/1, and sum_k phi_hat_k(r + h_k beta) must equal Sigma_{phi_beta s} z of the
    LTAO path (Eq.15, covariance.dense_cos_direct) to rounding (pin ii)."""
    base = replace(get_config("cfg1"), n=8, D=4.0)
    d = base.D / base.n
    h = (0.0, 5000.0, 10000.0)
    step = d / 5000.0 / geo.ARCSEC                             # arcsec that move the footprint by one step at 5 km
    cfg = replace(base, h=h, frac=(0.5, 0.3, 0.2))
    s = _system(cfg)
    beta = (2 * step, -1 * step)                               # (2, -1) steps at 5 km, (4, -2) at 10 km
    n_m = lay.n_meta(s.n, s.d, h, s.h_gs, 4.5 * step)
    z = np.random.default_rng(3).standard_normal(s.Ns)
    layers = lay.layered_estimate(z, n_m, s.centres, s.d, s.dirs, s.h_gs, h, cfg.frac, cfg.r0, cfg.L0)
    got = lay.ray_trace(layers, s.phase_pts, s.d, s.h_gs, h, beta)
    want = s.dense_cos_direct(beta) @ z
    assert np.allclose(got, want, atol=1e-11 * np.abs(want).max())
    # a wrong sign of h_k beta, a transposed grid or a wrong centre does not survive this:
    bad = lay.ray_trace(layers, s.phase_pts, s.d, s.h_gs, h, (-beta[0], -beta[1]))
    assert np.abs(bad - want).max() > 1e-3 * np.abs(want).max()
    # generic direction: bilinear interpolation of a smooth field, close but not equal
    b2 = (1.3 * step, 0.4 * step)
    e = lay.ray_trace(layers, s.phase_pts, s.d, s.h_gs, h, b2) - s.dense_cos_direct(b2) @ z
    assert 0 < np.linalg.norm(e) < 0.05 * np.linalg.norm(want)


def test_lgs_on_axis_layers_are_the_xi_prime_of_eq17():
    """LGS, beta = 0: the LTAO new grid of Eq.16 (L189) is centred on the axis like the layer grid, so with n_m = n' the
    layer covariance is Xi'_k itself and I'_k of the LTAO path ray-traces it: sum_k I'_k phi_hat_k = Eq.17 (L195)."""
    cfg = small_lgs_config(n=8, n_gs=3, n_layers=3, targets=((0.0, 0.0),))
    s = OracleSystem(cfg)
    z = np.random.default_rng(5).standard_normal(s.Ns)
    _, parts = cov.dense_cos_interpolated(s.phase_pts, s.centres, s.d, s.dirs, s.h_gs, (0.0, 0.0), cfg.h, cfg.frac,
                                          cfg.r0, cfg.L0, s.n_p, return_layers=True)
    layers = lay.layered_estimate(z, s.n_p, s.centres, s.d, s.dirs, s.h_gs, cfg.h, cfg.frac, cfg.r0, cfg.L0)
    for k, (Ik, xi) in enumerate(parts):
        assert np.allclose(layers[k].ravel(), xi @ z, atol=1e-12)
    assert np.allclose(lay.ray_trace(layers, s.phase_pts, s.d, s.h_gs, cfg.h, (0.0, 0.0)), s.Cos[0] @ z, atol=1e-11)
    # a larger grid contains the smaller one in its centre
    big = lay.layered_estimate(z, s.n_p + 4, s.centres, s.d, s.dirs, s.h_gs, cfg.h, cfg.frac, cfg.r0, cfg.L0)
    assert np.allclose(big[:, 2:-2, 2:-2], layers, atol=1e-12)


@pytest.mark.parametrize("lgs", [False, True])
def test_layer_product_is_2rbt_with_the_on_axis_generators(lgs):
    """L199: "... with the 2RBT formulation": Sigma_{phi_k s} z from positions == the Toeplitz product with the
    generators xi'_k of L193 taken at beta = 0 on the n_m grid (toeplitz.cos_generators), by zero-padded 2-D FFTs."""
    cfg = small_lgs_config(n=6, n_gs=3, n_layers=3) if lgs else replace(get_config("cfg1"), n=6, D=3.0)
    s = _system(cfg)
    c = cfg
    n_m = lay.n_meta(s.n, s.d, c.h, s.h_gs, 25.0)
    z = np.random.default_rng(7).standard_normal(s.Ns)
    want = lay.layered_estimate(z, n_m, s.centres, s.d, s.dirs, s.h_gs, c.h, c.frac, c.r0, c.L0)
    xi = tz.cos_generators(s.n, n_m, s.d, s.dirs, s.h_gs, (0.0, 0.0), c.h, c.frac, c.r0, c.L0)
    zf = np.zeros((s.N, 2, s.n * s.n))
    zf[:, :, s.sub_idx] = z.reshape(s.N, 2, s.nv)
    zf = zf.reshape(s.N, 2, s.n, s.n)
    P = n_m + s.n - 1
    for k in range(len(c.h)):
        g = np.zeros((n_m, n_m))
        for j in range(s.N):
            for b in range(2):
                g += tz.rbt_mvm_fft2(xi[k, j, b], zf[j, b], n_m, P)
        assert np.allclose(g, want[k], atol=1e-10 * np.abs(want).max())
