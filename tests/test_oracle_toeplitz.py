"""Pins for oracle/toeplitz.py: the paper's index maps (Eq.18-26) on brute-force tiny cases,
dense-from-positions == generator/Toeplitz == zero-padded 2-D FFT, printed closed forms."""
import os

import numpy as np
import pytest

from oracle import covariance as cov
from oracle import geometry as geo
from oracle import toeplitz as tz
from oracle.system import OracleSystem
from tomo_inputs import get_config
from tomo_inputs.configs import small_lgs_config


@pytest.mark.parametrize("m,n", [(4, 4), (5, 4), (7, 3), (3, 6), (9, 8)])
def test_paper_index_maps_exact(m, n):
    rng = np.random.default_rng(m * 100 + n)
    tab = rng.standard_normal((m + n - 1, m + n - 1))

    def g(a, b):                         # any function of the lags (i-i', j-j')
        return tab[a + n - 1, b + n - 1]
    T = tz.rbt_dense(g, m, n)
    x = rng.standard_normal(n * n)
    y = tz.rbt_mvm_paper(tz.t_vector(g, m, n), x, m, n)
    assert np.allclose(y, T @ x, atol=1e-12)
    # S_1 has n^2 non-zeros, S_2 m^2, all indices distinct and inside the vector (L221, L247)
    mu_1 = {tz.mu1(i, j, m, n) for i in range(n) for j in range(n)}
    mu_2 = {tz.mu2(i, j, m, n) for i in range(m) for j in range(m)}
    assert len(mu_1) == n * n and len(mu_2) == m * m
    assert min(mu_1) >= 0 and max(mu_1) < (m + n - 1) ** 2
    assert min(mu_2) >= 0 and max(mu_2) < (m + n - 1) ** 2


@pytest.mark.parametrize("P", [15, 16, 20])
def test_fft2_form_equals_dense(P):
    n = 8
    rng = np.random.default_rng(P)
    theta = rng.standard_normal((2 * n - 1, 2 * n - 1))
    x = rng.standard_normal((n, n))
    # y[p] = sum_q theta(q - p) x[q]
    y = np.zeros((n, n))
    for py in range(n):
        for px in range(n):
            for qy in range(n):
                for qx in range(n):
                    y[py, px] += theta[qy - py + n - 1, qx - px + n - 1] * x[qy, qx]
    assert np.allclose(tz.rbt_mvm_fft2(theta, x, n, P), y, atol=1e-11)


def test_dense_from_positions_is_2rbt_lgs():
    """L150/L158: with all LGS at one altitude every block is 2RBT -- the generator built from
    lags reproduces the dense matrix built from positions, entry by entry."""
    cfg = small_lgs_config(n=6, n_gs=3, n_layers=3, D=3.0)
    s = OracleSystem(cfg, build_cos=False)
    th = s.generators()
    n, nv, N = s.n, s.nv, s.N
    C = s.Css.reshape(N, 2, nv, N, 2, nv)
    for i in range(N):
        for j in range(N):
            for a in range(2):
                for b in range(2):
                    blk = th[i, a, j, b][(s.iy[None, :] - s.iy[:, None]) + n - 1,
                                         (s.ix[None, :] - s.ix[:, None]) + n - 1]
                    assert np.allclose(C[i, a, :, j, b, :], blk, atol=1e-10)
    # block-transpose symmetry Theta_(i,a),(j,b)(l) = Theta_(j,b),(i,a)(-l)
    assert np.allclose(th[0, 0, 1, 1], th[1, 1, 0, 0][::-1, ::-1], atol=1e-10)


def test_css_fft_product_equals_dense_and_directsum():
    from oracle import directsum
    cfg = small_lgs_config(n=6, n_gs=3, n_layers=3, D=3.0)
    s = OracleSystem(cfg, build_cos=False)
    th = s.generators()
    rng = np.random.default_rng(3)
    x = rng.standard_normal(s.Ns)
    ref = s.Css @ x
    for P in (11, 12, 16):
        spec = tz.css_spectra(th, s.n, P)
        xf = np.zeros((s.N, 2, s.n * s.n))
        xf[:, :, s.sub_idx] = x.reshape(s.N, 2, s.nv)
        y = tz.css_mvm_fft(spec, xf.reshape(s.N, 2, s.n, s.n), s.n, P)
        y = y.reshape(s.N, 2, -1)[:, :, s.sub_idx].ravel()
        assert np.allclose(y, ref, atol=1e-9)
    assert np.allclose(directsum.css_mvm(th, s.ix, s.iy, x), ref, atol=1e-9)
    # spectra: Hermitian across the block transpose, real on the block diagonal
    spec = tz.css_spectra(th, s.n, 12)
    assert np.allclose(spec[0, 0, 1, 1], np.conj(spec[1, 1, 0, 0]), atol=1e-9)
    full = np.fft.fft2(tz.embed_generator(th[2, 1, 2, 1], s.n, s.n, 12))
    assert np.abs(full.imag).max() < 1e-9


def test_matrix_free_operator_equals_dense_operator():
    cfg = small_lgs_config(n=6, n_gs=3, n_layers=2, D=3.0)
    sd = OracleSystem(cfg, build_cos=False)
    sm = OracleSystem(cfg, dense=False, build_cos=False)
    v = np.random.default_rng(5).standard_normal(sd.Ns)
    assert np.allclose(sm.apply_A(v), sd.apply_A(v), atol=1e-9)


def _golden():
    rows = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_closed_forms.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, val, tol, _ = [s.strip() for s in line.split("|", 3)]
            rows[name] = (float(val), float(tol))
    return rows


def test_printed_closed_forms():
    g = _golden()
    n, N, K, a = 80, 6, 9, 5.0

    def close(name, val):
        ref, tol = g[name]
        # the paper prints one significant digit: compare after rounding to it
        assert abs(val / ref - 1) < max(tol, 0.0), (name, val, ref)
    close("compression_css_n80", tz.compression_css(n))
    close("compression_cos_ngs_n80", tz.compression_cos_ngs(n))
    n_p = int(round(1.2 * n))
    # n'_k "roughly n h_lgs/(h_lgs-h_k)" (L179), layers evenly spread up to 16 km (Fig.8 caption)
    npk = [int(np.ceil(n * 90.0 / (90.0 - hk))) for hk in np.linspace(0, 16, K)]
    close("compression_cos_lgs_n80", tz.compression_cos_lgs(n, npk, N, K))
    close("reduction_css_n80", tz.reduction_css(n, N, a))
    close("reduction_cos_ngs_n80", tz.ops_cos_ngs(n, N, a) / (2 * N * (n + 1) ** 2 * n ** 2))
    close("reduction_cos_lgs_n80", tz.ops_cos_lgs(n, n_p, N, K, a) / (2 * N * (n + 1) ** 2 * n ** 2))
    # unique-element counts (L150, L177, L193)
    assert (2 * n - 1) ** 2 == 25281
    assert abs(tz.ops_css(74, 6, 5.0) / 4.32e9 - 40.6e6 / 4.32e9) < 1e-3


def test_rows_from_positions_pin_the_generator_and_direct_sum_routes():
    """OracleSystem.css_rows_explicit (rows of W Sigma_ss W^T straight from subaperture positions, what the full-size GPU
    tests sample) = the dense matrix = the generator / direct-sum route used when the dense matrix does not fit."""
    import numpy as np
    from oracle.system import OracleSystem
    from tomo_inputs.configs import small_lgs_config
    cfg = small_lgs_config(n=10, n_gs=3, n_layers=3)
    dense = OracleSystem(cfg, build_cos=False)
    free = OracleSystem(cfg, dense=False, build_cos=False)
    rows = [0, 17, dense.nv + 3, 5 * dense.nv - 1]
    R = free.css_rows_explicit(rows)
    assert np.allclose(R, dense.Css[rows], rtol=0, atol=1e-12 * np.abs(dense.Css).max())
    u = np.random.default_rng(0).standard_normal(dense.Ns)
    assert np.allclose(R @ u, free.css_unprojected(u)[rows], rtol=1e-12, atol=1e-10)
