"""Pins for the phase-slope projection (Eq.13, Eq.15-17, Eq.31-32)."""
from dataclasses import replace

import numpy as np

from oracle import covariance as cov
from oracle import geometry as geo
from oracle import toeplitz as tz
from oracle.system import OracleSystem
from tomo_inputs import get_config, screens
from tomo_inputs.configs import small_lgs_config


def test_n_prime_values():
    # reading G19; sizes quoted in DESIGN.md for the configs
    assert geo.n_prime(20, 1 - 16000 / 90e3) == 27
    assert geo.n_prime(74, 1 - 25000 / 90e3) == 105
    assert [geo.n_prime(n, 1 - 25000 / 90e3) for n in (16, 32, 64, 96, 128)] == [25, 47, 91, 135, 179]
    assert geo.n_prime(8, 1.0) == 9


def test_valid_counts():
    for n, nv, nvp in [(8, 52, 69), (16, 208, 241), (20, 316, 357), (74, 4304, 4453)]:
        sm = geo.subap_mask(n, 1.0)
        assert sm.sum() == nv and geo.phase_mask(sm).sum() == nvp


def test_ground_layer_interpolated_equals_direct():
    cfg = replace(small_lgs_config(n=8, n_gs=3, n_layers=1), h=(0.0,), frac=(1.0,))
    s = OracleSystem(cfg)
    direct = s.dense_cos_direct(cfg.targets[0])
    assert np.allclose(s.Cos[0], direct, atol=1e-10)
    # and the bilinear matrix is a pure selection there
    I0 = cov.bilinear_matrix(s.phase_pts, s.d, s.n_p)
    assert set(np.unique(I0)) <= {0.0, 1.0} and np.all(I0.sum(axis=1) == 1.0)


def test_bilinear_rows():
    cfg = small_lgs_config(n=8, n_gs=3, n_layers=3)
    s = OracleSystem(cfg, build_cos=False)
    for hk in cfg.h:
        dk = geo.cone_factor(hk, s.h_gs) * s.d
        Ik = cov.bilinear_matrix(s.phase_pts, dk, s.n_p)
        assert np.allclose(Ik.sum(axis=1), 1.0)
        assert (Ik != 0).sum(axis=1).max() <= 4 and Ik.min() >= 0
        # reproduces linear functions of position exactly
        g1 = (np.arange(s.n_p) - (s.n_p - 1) / 2.0) * dk
        GX, GY = np.meshgrid(g1, g1, indexing="xy")
        assert np.allclose(Ik @ (2 * GX - 3 * GY).ravel(), 2 * s.phase_pts[:, 0] - 3 * s.phase_pts[:, 1])


def test_interpolated_close_to_direct_and_reported():
    cfg = small_lgs_config(n=10, n_gs=3, n_layers=3, targets=((5.0, -3.0),))
    s = OracleSystem(cfg)
    direct = s.dense_cos_direct(cfg.targets[0])
    rel = np.linalg.norm(s.Cos[0] - direct) / np.linalg.norm(direct)
    assert 0 < rel < 0.02          # an approximation (L392), small but not zero


def test_fft_path_equals_dense_interpolated():
    """Eq.32: sum_k I'_k S_2 F^-1{sum_j xi'~ . zeta~} == dense sum_k I'_k Xi'_k, off-axis target."""
    cfg = small_lgs_config(n=8, n_gs=3, n_layers=3, targets=((7.0, 4.0),))
    s = OracleSystem(cfg)
    c = cfg
    beta = c.targets[0]
    z = np.random.default_rng(1).standard_normal(s.Ns)
    xi = tz.cos_generators(s.n, s.n_p, s.d, s.dirs, s.h_gs, beta, c.h, c.frac, c.r0, c.L0)
    P = s.n_p + s.n - 1 + 2
    zf = np.zeros((s.N, 2, s.n * s.n))
    zf[:, :, s.sub_idx] = z.reshape(s.N, 2, s.nv)
    zf = zf.reshape(s.N, 2, s.n, s.n)
    out = np.zeros(s.nvp)
    for k, hk in enumerate(c.h):
        g = np.zeros((s.n_p, s.n_p))
        for j in range(s.N):
            for b in range(2):
                g += tz.rbt_mvm_fft2(xi[k, j, b], zf[j, b], s.n_p, P)
        Ik = cov.bilinear_matrix(s.phase_pts, geo.cone_factor(hk, s.h_gs) * s.d, s.n_p)
        out += Ik @ g.ravel()
    assert np.allclose(out, s.Cos[0] @ z, atol=1e-9)
    # the matrix-free (direct-sum) route of system.py agrees too
    sm = OracleSystem(cfg, dense=False, build_cos=False)
    assert np.allclose(sm.cos_matrix_free(z, 0), s.Cos[0] @ z, atol=1e-9)
    assert np.allclose(sm.reconstruct(z, 0), s.reconstruct(z, 0), atol=1e-9)


def test_ngs_eq31_fft_equals_dense():
    s = OracleSystem(get_config("cfg1"))
    c = s.cfg
    z = np.random.default_rng(2).standard_normal(s.Ns)
    m = s.n + 1
    # layer-summed generator on the (n+1) grid: lag l = q - p, Delta = d l + d/2 + h(alpha - beta)
    xi = tz.cos_generators(s.n, m, s.d, s.dirs, s.h_gs, c.targets[0], c.h, c.frac, c.r0, c.L0).sum(axis=0)
    zf = np.zeros((s.N, 2, s.n * s.n))
    zf[:, :, s.sub_idx] = z.reshape(s.N, 2, s.nv)
    zf = zf.reshape(s.N, 2, s.n, s.n)
    g = np.zeros((m, m))
    for j in range(s.N):
        for b in range(2):
            g += tz.rbt_mvm_fft2(xi[j, b], zf[j, b], m, 16)
    assert np.allclose(g.ravel()[s.ph_idx], s.Cos[0] @ z, atol=1e-9)


def test_end_to_end_mmse_reduces_error_and_pins_signs():
    for cfg in (get_config("cfg1"), small_lgs_config(n=10, n_gs=3, n_layers=3)):
        s = OracleSystem(cfg)
        inp = screens.generate(cfg, s.sigma2)
        sl = inp["slopes"][0].ravel()
        zd = s.solve_direct(sl)
        phi = s.reconstruct(zd)
        truth = s.Mphi @ inp["truth"][0, 0]
        err = np.linalg.norm(phi - truth) / np.linalg.norm(truth)
        assert err < 0.6, err
        assert np.corrcoef(phi, truth)[0, 1] > 0.8
        assert np.linalg.norm(-phi - truth) / np.linalg.norm(truth) > 1.2     # flipped sign fails
