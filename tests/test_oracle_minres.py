"""Pins for oracle/solver.py:minres (PAPER.md S2.G L337, L426: the paper's solver for the Toeplitz method).

The paper prints no pseudo-code, so the oracle is pinned to what defines the method: the k-th iterate minimises
|b - A x| over x0 + K_k(A, r0) (brute force: explicit Krylov basis + dense least squares), phibar_k is that
minimum, the residual norm never increases, the iterates reach the direct solution, and an independent library
routine (scipy.sparse.linalg.minres) produces the same iterates.
"""
import numpy as np
import pytest
import scipy.sparse.linalg as spla

from oracle import solver
from oracle.system import OracleSystem
from tomo_inputs import get_config, screens
from tomo_inputs.configs import small_lgs_config


def _krylov_minimiser(A, b, x0, k):
    r0 = b - A @ x0
    K = np.empty((len(b), k))
    v = r0.copy()
    for j in range(k):
        K[:, j] = v / np.linalg.norm(v)
        v = A @ K[:, j]
    Q, _ = np.linalg.qr(K)                                   # same span, well conditioned
    y, *_ = np.linalg.lstsq(A @ Q, r0, rcond=None)
    return x0 + Q @ y


@pytest.mark.parametrize("kind", ["spd", "indefinite"])
def test_minres_is_the_krylov_least_squares_minimiser(kind):
    rng = np.random.default_rng(7)
    n = 14
    B = rng.standard_normal((n, n))
    A = B @ B.T + 0.5 * np.eye(n) if kind == "spd" else (B + B.T)
    b = rng.standard_normal(n)
    x0 = rng.standard_normal(n) * 0.3
    for k in range(1, 9):
        x, hist = solver.minres(lambda v: A @ v, b, k, x0=x0)
        xk = _krylov_minimiser(A, b, x0, k)
        assert np.linalg.norm(x - xk) <= 1e-9 * np.linalg.norm(xk)
        assert abs(hist[k] - np.linalg.norm(b - A @ x)) <= 1e-10 * hist[0]      # phibar_k = |b - A x_k|
        assert hist.shape == (k + 1,) and abs(hist[0] - np.linalg.norm(b - A @ x0)) < 1e-12


def test_minres_matches_scipy_iterates():
    rng = np.random.default_rng(11)
    n = 40
    B = rng.standard_normal((n, n))
    A = B @ B.T + np.eye(n)
    b = rng.standard_normal(n)
    for k in (1, 2, 5, 12, 25):
        x, _ = solver.minres(lambda v: A @ v, b, k)
        xs, _ = spla.minres(A, b, rtol=0.0, maxiter=k)
        assert np.linalg.norm(x - xs) <= 1e-9 * np.linalg.norm(xs)


def test_minres_exact_after_dimension_steps_and_freezes():
    rng = np.random.default_rng(3)
    n = 6
    B = rng.standard_normal((n, n))
    A = B @ B.T + np.eye(n)
    b = rng.standard_normal(n)
    x, hist = solver.minres(lambda v: A @ v, b, n + 4)           # Krylov space exhausted after n steps
    assert np.linalg.norm(A @ x - b) < 1e-9 * np.linalg.norm(b)
    assert np.all(np.isfinite(hist)) and np.all(np.isfinite(x))
    x0, h0 = solver.minres(lambda v: A @ v, np.zeros(n), 3)      # zero rhs: nothing to do
    assert np.all(x0 == 0) and np.all(h0 == 0)


def test_minres_on_cfg1_monotone_and_converges_to_direct():
    s = OracleSystem(get_config("cfg1"), build_cos=False)
    sl = screens.generate(s.cfg, s.sigma2)["slopes"][0].ravel()
    zd = s.solve_direct(sl)
    x, hist, st = s.solve_minres(sl, s.Ns, record=True)
    assert np.linalg.norm(x - zd) / np.linalg.norm(zd) < 1e-8
    assert np.all(np.diff(hist[:120]) <= 1e-12 * hist[0])         # residual norm never increases (CG's does, G17)
    b = s.rhs(sl)
    for k in (1, 5, 20, 50):
        assert abs(hist[k] - np.linalg.norm(b - s.A @ st[k - 1]["x"])) < 1e-8 * hist[0]
    # MINRES residual <= CG residual at every count (it minimises what CG only bounds)
    _, hcg = s.solve_cg(sl, 60)
    assert np.all(hist[:61] <= hcg * (1 + 1e-9))


def test_minres_singular_system_stays_in_range():
    """Mode removal makes A singular (null space = span Z, G14); b = M s is consistent, so MINRES converges to A^+ b
    and the iterates keep zero mean slope per WFS."""
    cfg = small_lgs_config(n=6, n_gs=3, n_layers=2, D=3.0)
    s = OracleSystem(cfg, build_cos=False)
    sl = screens.generate(cfg, s.sigma2)["slopes"][0].ravel()
    zd = s.solve_direct(sl)
    x, hist = s.solve_minres(sl, 150)
    assert np.linalg.norm(x - zd) / np.linalg.norm(zd) < 1e-7
    assert np.abs(x.reshape(s.N, 2, s.nv).mean(axis=2)).max() < 1e-9 * np.abs(x).max()
    # warm start from a perturbed solution converges in fewer iterations (L428, L506)
    x0 = s.project_slopes(zd + 0.01 * np.random.default_rng(0).standard_normal(zd.shape) * np.abs(zd).max())
    _, hw = s.solve_minres(sl, 30, x0=x0)
    assert hw[0] < hist[0] and hw[30] < hist[30]
