"""Pins for the 2 x 2 block-diagonal noise covariance of elongated LGS spots in the oracle and for the
seeded recipe that stands in for it (tomo_inputs.screens.elongated_noise_blocks)."""
import numpy as np

from oracle.system import OracleSystem
from tomo_inputs import screens
from tomo_inputs.configs import small_lgs_config


def test_blocks_are_spd_reduce_to_diagonal_and_follow_the_launch_geometry():
    cfg = small_lgs_config(n=8, n_gs=3, n_layers=2)
    sxx, syy, sxy = screens.elongated_noise_blocks(cfg, 2.0, elongation=3.0)
    assert np.all(sxx * syy - sxy ** 2 > 0) and np.all(sxx >= 2.0) and np.all(syy >= 2.0)
    # smaller eigenvalue = sigma2 (across the elongation), larger = sigma2 (1 + elong (|e|/D)^2) (along it)
    tr, det = sxx + syy, sxx * syy - sxy ** 2
    lam_min = 0.5 * (tr - np.sqrt(tr ** 2 - 4 * det))
    assert np.allclose(lam_min, 2.0, rtol=1e-12)
    assert (0.5 * (tr + np.sqrt(tr ** 2 - 4 * det))).max() <= 2.0 * (1 + 3.0 * 1.0) + 1e-9      # |e| <= D
    z = screens.elongated_noise_blocks(cfg, 2.0, elongation=0.0)
    assert np.all(z[0] == 2.0) and np.all(z[1] == 2.0) and np.all(z[2] == 0.0)
    # sample covariance of the drawn noise -> the blocks
    zero = np.zeros((4000, cfg.n_wfs, 2, sxx.shape[1]))
    nz = screens.add_block_noise(cfg, zero, (sxx, syy, sxy))
    i, q = 1, 5
    c = np.cov(nz[:, i, 0, q], nz[:, i, 1, q])
    assert np.allclose(c, [[sxx[i, q], sxy[i, q]], [sxy[i, q], syy[i, q]]], rtol=0.12, atol=0.1)


def test_oracle_operator_with_blocks():
    cfg = small_lgs_config(n=6, n_gs=2, n_layers=2, D=3.0)
    base = OracleSystem(cfg, build_cos=False)
    blocks = screens.elongated_noise_blocks(cfg, base.sigma2, elongation=2.0)
    s = OracleSystem(cfg, build_cos=False, noise_blocks=blocks)
    # Sigma_eta: symmetric, SPD, 3 non-zero diagonals per subaperture pair (L110: "only 3 central diagonals")
    assert np.allclose(s.Cnn, s.Cnn.T) and np.linalg.eigvalsh(s.Cnn).min() > 0
    assert np.count_nonzero(s.Cnn) == 4 * s.N * s.nv - np.count_nonzero(np.asarray(blocks[2]) == 0) * 2
    # the operator differs from the diagonal-noise one exactly by M (Sigma_eta - sigma^2 I) M
    d = s.A - base.A
    assert np.allclose(d, s.Ms @ (s.Cnn - base.sigma2 * np.eye(s.Ns)) @ s.Ms.T, atol=1e-10)
    # x-y coupling: a pure x-slope vector of WFS 0 produces y-slope output through the noise term alone
    v = np.zeros(s.Ns); v[3] = 1.0
    out = (s.Cnn @ v).reshape(s.N, 2, s.nv)
    assert out[0, 1, 3] == blocks[2][0, 3] and out[0, 0, 3] == blocks[0][0, 3] and np.count_nonzero(out) == 2
    # zero elongation = the diagonal system
    s0 = OracleSystem(cfg, build_cos=False, noise_blocks=screens.elongated_noise_blocks(cfg, base.sigma2, elongation=0.0))
    assert np.allclose(s0.A, base.A, atol=1e-12)
    # CG still converges to the direct solve
    sl = screens.generate(cfg, base.sigma2)["slopes"][0].ravel()
    x, h = s.solve_cg(sl, s.Ns)
    assert h[-1] < 1e-9 * h[0]
    zd = s.solve_direct(sl)
    assert np.linalg.norm(x - zd) / np.linalg.norm(zd) < 1e-8
