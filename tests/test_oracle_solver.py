"""Pins for oracle/projectors.py and oracle/solver.py (Eq.36, Eq.12, S2.G L337)."""
import numpy as np

from oracle import projectors as prj
from oracle import solver
from oracle.system import OracleSystem
from tomo_inputs import get_config, screens
from tomo_inputs.configs import small_lgs_config


def test_projector_identities():
    cfg = small_lgs_config(n=8, n_gs=2, n_layers=2)
    s = OracleSystem(cfg, build_cos=False)
    for nr in (2, 3):
        Z = prj.slope_modes(s.centres, nr)
        M = prj.removal_matrix(Z)
        assert np.allclose(M @ M, M, atol=1e-12)
        assert np.allclose(M, M.T, atol=1e-12)
        assert np.allclose(M @ Z, 0, atol=1e-12)
        assert abs(np.trace(M) - (2 * s.nv - nr)) < 1e-9
    v = np.random.default_rng(0).standard_normal(s.Ns)
    u = (s.Ms @ v).reshape(s.N, 2, s.nv)
    assert np.abs(u.mean(axis=2)).max() < 1e-12          # zero mean x / y slope per WFS
    Zp = prj.phase_modes(s.phase_pts, 2)
    Mp = prj.removal_matrix(Zp)
    assert np.allclose(Mp @ Zp, 0, atol=1e-10) and Zp.shape[1] == 3


def test_null_space_dimension():
    cfg = small_lgs_config(n=6, n_gs=3, n_layers=2, D=3.0)
    s = OracleSystem(cfg, build_cos=False)
    w = np.linalg.eigvalsh(s.A)
    nz = int(np.sum(np.abs(w) < 1e-8 * w.max()))
    assert nz == 2 * s.N                                  # n_remove * N zero eigenvalues
    assert w.min() > -1e-8 * w.max()


def test_cg_converges_to_direct_cfg1():
    s = OracleSystem(get_config("cfg1"), build_cos=False)
    sl = screens.generate(s.cfg, s.sigma2)["slopes"][0].ravel()
    zd = s.solve_direct(sl)
    assert np.allclose(s.A @ zd, s.rhs(sl), atol=1e-8)
    x, hist, st = s.solve_cg(sl, s.Ns, record=True)
    assert np.linalg.norm(x - zd) / np.linalg.norm(zd) < 1e-8
    # A-norm of the error decreases monotonically (textbook CG property) while it is resolvable
    errs = [float((t["x"] - zd) @ s.A @ (t["x"] - zd)) for t in st[:60]]
    assert all(e1 <= e0 * (1 + 1e-9) for e0, e1 in zip(errs, errs[1:]))
    assert hist.shape == (s.Ns + 1,) and abs(hist[0] - np.linalg.norm(s.rhs(sl))) < 1e-9
    # teacher-forced identities: r_{k+1} = r_k - alpha q, p_{k+1} = r_{k+1} + beta p_k
    t0, t1 = st[3], st[4]
    assert np.allclose(t1["r"], t0["r"] - t0["alpha"] * t0["q"], atol=1e-10)
    assert np.allclose(t1["p"], t1["r"] + t0["beta"] * t0["p"], atol=1e-10)
    assert abs(t0["alpha"] - t0["rho"] / (t0["p"] @ t0["q"])) < 1e-12


def test_cg_singular_system_stays_in_range():
    cfg = small_lgs_config(n=8, n_gs=3, n_layers=3)
    s = OracleSystem(cfg, build_cos=False)
    sl = screens.generate(cfg, s.sigma2)["slopes"][0].ravel()
    zd = s.solve_direct(sl)
    # (run far beyond convergence the fixed-count recurrence drifts into range(Z): stop at 150)
    x, hist = s.solve_cg(sl, 150)
    assert np.linalg.norm(x - zd) / np.linalg.norm(zd) < 1e-6
    assert np.abs(x.reshape(s.N, 2, s.nv).mean(axis=2)).max() < 1e-9 * np.abs(x).max() + 1e-12


def test_warm_start_and_matrix_free_cg():
    cfg = small_lgs_config(n=6, n_gs=2, n_layers=2, D=3.0)
    sd = OracleSystem(cfg, build_cos=False)
    sm = OracleSystem(cfg, dense=False, build_cos=False)
    sl = screens.generate(cfg, sd.sigma2)["slopes"][0].ravel()
    xd, hd = sd.solve_cg(sl, 15)
    xm, hm = sm.solve_cg(sl, 15)
    assert np.allclose(hd, hm, rtol=1e-8)
    assert np.allclose(xd, xm, atol=1e-9 * np.abs(xd).max())
    xw, hw = sd.solve_cg(sl, 5, x0=xd)
    assert hw[0] < hd[0] and abs(hw[0] - hd[-1]) < 1e-6 * hd[0]
