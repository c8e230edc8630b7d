"""Parity of the MINRES path (tomo_solve_minres through the C ABI) with the oracle's textbook MINRES
(oracle/solver.py:minres; PAPER.md S2.G L337, L426: the paper's solver for the Toeplitz method).

The product kernels are the CG path's (gate P-a).  MINRES trajectories share CG's Lanczos process and so its
reproducibility horizon; the gates mirror P-c / P-d / P-e:
  M-c  free-running fp32:  phibar_k and x_k within 1e-3 of the fp64 oracle up to the horizon at which an fp32 CPU emulation of
                           the same algorithm leaves 1e-3 (minus 2); the full-count deviation is printed
  M-d  converged:          wavefront vs the direct solve <= 1e-3 once the oracle's MINRES is below 1e-6
  M-e  fp64 instantiation: phibar_k within 1e-6 and x_k within 1e-5 of the oracle at every k up to the horizon at which
                           two fp64 oracle runs (rhs perturbed by 1e-15) agree to 1e-4 -- every recurrence of every step
  plus: warm start, zero iterations, batch frames = single solves bitwise, monotone residual, MINRES <= CG residual.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1806_07938_b200 import tomo  # noqa: E402
from test_gpu_parity import TOL_TRAJ, _horizon, dev, f32, make_plan, rel, solvers, system  # noqa: E402

pytestmark = pytest.mark.gpu


def _gpu_minres(pl, s, n_it, x0=None, want_x=True):
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve_minres(dev(s), d_w, 1, n_it, x0=None if x0 is None else dev(x0))
    z = torch.empty(pl.slopes_len, dtype=torch.float32, device="cuda")
    pl.get_zeta(z)
    torch.cuda.synchronize()
    return d_w.cpu().numpy(), z.cpu().numpy(), pl.residuals(1, n_it)[0]


@solvers
@pytest.mark.parametrize("name", ["cfg1", "small_lgs", "small_odd_focus", "cfg2"])
def test_minres_free_running_fp32_tracks_oracle_up_to_the_fp32_horizon(name, solver):
    cfg, _, osys, data = system(name)
    n_it = cfg.n_iter
    s = f32(data["slopes"][0].ravel())
    _, h64 = osys.solve_minres(s, n_it)
    _, h32 = osys.solve_minres(s, n_it, dtype=np.float32)
    k_star = max(_horizon(h32, h64) - 2, 3)
    pl = make_plan(name, solver=solver)
    _, _, hg = _gpu_minres(pl, s, n_it)
    d = np.abs(hg / h64 - 1.0)
    assert d[:k_star + 1].max() <= TOL_TRAJ, (name, k_star, d[:k_star + 1].max())
    assert np.all(np.diff(hg) <= 1e-6 * hg[0])                      # the residual norm never increases
    _, zk, _ = _gpu_minres(pl, s, k_star)
    assert rel(zk, osys.solve_minres(s, k_star)[0]) <= TOL_TRAJ, (name, k_star)
    print(f"[M-c {name}] fp32 horizon k*={k_star}; deviation of phibar_k at the full count {n_it}: {d[-1]:.2e}")
    pl.close()


@solvers
@pytest.mark.parametrize("name", ["cfg1", "small_lgs", "small_fried", "ngs_offaxis", "cfg2"])
def test_minres_converged_solution_matches_direct_solve(name, solver):
    cfg, _, osys, data = system(name)
    s = f32(data["slopes"][0].ravel())
    zeta = osys.solve_direct(s)
    _, h = osys.solve_minres(s, 1000)
    n_it = int(np.flatnonzero(h / h[0] < 1e-6)[0])
    pl = make_plan(name, solver=solver)
    w, _, hg = _gpu_minres(pl, s, n_it)
    got = w.reshape(len(cfg.targets), -1)
    for t in range(len(cfg.targets)):
        e = rel(got[t], osys.reconstruct(zeta, t))
        assert e <= 1e-3, (name, t, n_it, e)
    pl.close()


@solvers
@pytest.mark.parametrize("name", ["cfg1", "small_lgs", "small_odd_focus", "cfg2"])
def test_minres_fp64_instantiation_tracks_every_step(name, solver):
    cfg, _, osys, data = system(name)
    n_it = cfg.n_iter
    s = f32(data["slopes"][0].ravel())
    _, h_a, st = osys.solve_minres(s, n_it, record=True)
    _, h_b = osys.solve_minres(s * (1.0 + 1e-15 * np.cos(np.arange(s.size))), n_it)
    k_rep = max(min(_horizon(h_b, h_a, tol=1e-4) - 2, n_it), 3)
    pl = make_plan(name, precision=tomo.TOMO_F64, solver=solver)
    _, _, hg = _gpu_minres(pl, s, k_rep)
    assert np.abs(hg / h_a[:k_rep + 1] - 1.0).max() <= 1e-6, (name, k_rep, np.abs(hg / h_a[:k_rep + 1] - 1.0).max())
    for k in sorted({1, 2, 3, k_rep // 2, k_rep}):
        _, zk, _ = _gpu_minres(pl, s, k)
        e = rel(zk, st[k - 1]["x"])
        assert e <= 1e-5, (name, k, e)                               # the ABI returns x in fp32: 6e-8 rounding
    print(f"[M-e {name}] two fp64 oracle runs agree to k={k_rep}; gated there")
    pl.close()


@solvers
def test_minres_warm_start_zero_iterations_batch_and_cg_comparison(solver):
    cfg, _, osys, data = system("small_lgs")
    pl = make_plan("small_lgs", max_batch=2, solver=solver)
    s2 = data["slopes"].reshape(2, -1)
    s = f32(s2[0])
    w, z, h = _gpu_minres(pl, s, 0)
    assert float(np.abs(w).max()) == 0.0 and float(np.abs(z).max()) == 0.0
    assert abs(h[0] / np.linalg.norm(osys.rhs(s)) - 1) < 1e-6
    # warm start (L428, L506) from the oracle's 6-iteration iterate
    x6 = osys.solve_minres(s, 6)[0]
    xo, ho = osys.solve_minres(s, 5, x0=f32(x6))
    _, zw, hw = _gpu_minres(pl, s, 5, x0=x6)
    assert np.abs(hw / ho - 1).max() <= TOL_TRAJ and rel(zw, xo) <= TOL_TRAJ
    # batch frames = single solves, bitwise
    n_it = 12
    d_w2 = torch.empty(2 * pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve_minres(dev(s2), d_w2, 2, n_it)
    torch.cuda.synchronize()
    h2 = pl.residuals(2, n_it)
    for f in range(2):
        d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
        pl.solve_minres(dev(s2[f]), d_w, 1, n_it)
        torch.cuda.synchronize()
        assert torch.equal(d_w, d_w2[f * pl.wavefront_len:(f + 1) * pl.wavefront_len])
        assert np.array_equal(pl.residuals(1, n_it)[0], h2[f])
    # MINRES minimises the residual CG only bounds: phibar_k <= |r_k| of the GPU's own CG at every k
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    h_cg = pl.residuals(1, n_it)[0]
    _, _, h_mr = _gpu_minres(pl, s, n_it)
    assert np.all(h_mr <= h_cg * (1 + 1e-5))
    pl.close()
