"""Parity of the CUDA path (through the C ABI) with the fp64 oracle on the same seeded inputs.

Gates (from north_star and SURVEY 8(c)):
  P-a  MVM and projection:       rel-L2 <= 1e-4 (fp32)
  P-b  teacher-forced CG step:   (x, r, p)_{k+1} rel-L2 <= 1e-4, alpha_k, beta_k to 1e-4, from the oracle's state
  P-c  free-running fp32 solve:  residual history and zeta within 1e-3 up to the horizon at which an fp32 CPU
                                 emulation of the same algorithm itself leaves 1e-3 (CG trajectories are chaotic
                                 beyond it, the deviation at the full count is reported, not gated)
  P-d  converged solve:          wavefront vs the direct (Cholesky / pseudo-inverse) solution <= 1e-3
  P-e  fp64 instantiation:       north_star's literal gate at the full iteration count (history and wavefront
                                 <= 1e-3) wherever two fp64 oracle runs agree with each other to 1e-4
"""
from dataclasses import replace

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.system import OracleSystem  # noqa: E402
from paper_1806_07938_b200 import tomo  # noqa: E402
from tomo_inputs import screens  # noqa: E402
from tomo_inputs.configs import WFS, get_config, small_lgs_config  # noqa: E402

from gates import assert_close, rel  # noqa: E402

pytestmark = pytest.mark.gpu

TOL_MVM = 1e-4
TOL_STEP = 1e-4
TOL_TRAJ = 1e-3


def dev(a, dtype=torch.float32):
    return torch.tensor(np.ascontiguousarray(a), dtype=dtype, device="cuda")


def f32(a):
    """The fp32-rounded input both sides see."""
    return np.asarray(a, dtype=np.float32).astype(np.float64)


def _case(name):
    if name == "cfg1":
        return get_config("cfg1"), "hudgin", None
    if name == "cfg2":
        return get_config("cfg2"), "hudgin", None
    if name == "small_lgs":          # two targets, one off-axis; ragged: n=10 -> P=20, P_os=24
        return small_lgs_config(n=10, n_gs=3, n_layers=3, targets=((5.0, -3.0), (0.0, 0.0))), "hudgin", None
    if name == "small_odd_focus":    # odd n (a single-row last pair), tip/tilt/focus removed, obstruction
        c = small_lgs_config(n=11, n_gs=3, n_layers=2, n_remove=3, targets=((0.0, 0.0),))
        return replace(c, obstruction=0.3), "hudgin", None
    if name == "small_fried":
        return small_lgs_config(n=8, n_gs=2, n_layers=2, targets=((2.0, 1.0),)), "fried", None
    if name == "small_fftmodel":     # FFT slope model (Eq.41-46): covariances by 2-D FFTs in the builder
        return small_lgs_config(n=8, n_gs=3, n_layers=2, targets=((3.0, -2.0),)), "fft", None
    if name == "ngs_offaxis":        # NGS, one WFS with tip/tilt removed and one without, off-axis target
        c = get_config("cfg1")
        return replace(c, wfs=(WFS(10.0, 0.0, float("inf"), 2), WFS(-10.0, 5.0)), targets=((3.0, 4.0),)), "hudgin", None
    raise KeyError(name)


_cache = {}


def system(name):
    if name not in _cache:
        cfg, model, _ = _case(name)
        osys = OracleSystem(cfg, model=model)
        data = screens.generate(cfg, osys.sigma2, n_frames=2)
        _cache[name] = (cfg, model, osys, data)
    return _cache[name]


def _oracle_fft_generators(cfg, osys):
    """Generators of the FFT slope model from the ORACLE (the continuous integrals of Eq.43 / Eq.46): css [C][C][2n-1][2n-1],
    cos [T][K][C][n'+n-1][n'+n-1] in the layout of tomo_plan_upload_kernels."""
    from oracle import toeplitz as tz
    n, N = cfg.n, len(cfg.wfs)
    css = tz.css_generators(n, cfg.d, osys.dirs, osys.h_gs, cfg.h, cfg.frac, cfg.r0, cfg.L0, "fft").reshape(2 * N, 2 * N, 2 * n - 1, 2 * n - 1)
    cos = []
    for beta in cfg.targets:
        xi = tz.cos_generators(n, osys.n_p, cfg.d, osys.dirs, osys.h_gs, beta, cfg.h, cfg.frac, cfg.r0, cfg.L0, "fft")
        cos.append(xi.reshape(xi.shape[0], 2 * N, xi.shape[-1], xi.shape[-1]))
    return css, np.stack(cos)


def make_plan(name, **kw):
    cfg, model, osys, _ = system(name)
    sm = {"fried": tomo.TOMO_FRIED, "fft": tomo.TOMO_FFTMODEL}.get(model, tomo.TOMO_HUDGIN)
    if model == "fft":
        # The oracle of the FFT slope model is the continuous integral; the library's builder evaluates it on a truncated
        # frequency grid (0.13 % of the slope variance off, gated in tests/test_host_builder.py).  The KERNELS are compared with
        # the oracle on the oracle's own generators (tomo_plan_upload_kernels takes them) and noise level;
        # test_fft_model_plan_from_the_builder below covers the plan the builder makes.
        if "fftgen" not in _cache:
            _cache["fftgen"] = _oracle_fft_generators(cfg, osys)
        css, cos = _cache["fftgen"]
        pl = tomo.TomoPlan(cfg, slope_model=sm, sigma2_wfs=[osys.sigma2] * len(cfg.wfs), css_gen=css, cos_gen=cos, **kw)
        assert pl.solver_in_use()[0] == kw.get("solver", tomo.TOMO_SOLVER_PERSISTENT), pl.solver_in_use()
        return pl
    pl = tomo.TomoPlan(cfg, slope_model=sm, **kw)
    # every plan of this file runs on the solver it asks for (default: the persistent kernel); none may fall back silently
    assert pl.solver_in_use()[0] == kw.get("solver", tomo.TOMO_SOLVER_PERSISTENT), pl.solver_in_use()
    s2, var = pl.noise()
    assert abs(s2[0] / osys.sigma2 - 1) < 1e-12 and abs(var / osys.slope_var - 1) < 1e-12
    sub, ph = pl.valid_index()
    assert np.array_equal(sub, osys.sub_idx) and np.array_equal(ph, osys.ph_idx)
    return pl


def test_fft_model_plan_from_the_builder_is_within_its_discretisation_error():
    """TOMO_FFTMODEL end to end with the BUILDER's generators (2-D FFTs on a grid cut at |f| < 2/w): product and converged
    wavefront within 1 % of the continuous-integral oracle (the generators are 0.13 % of the variance off; G29)."""
    cfg, model, osys, data = system("small_fftmodel")
    pl = tomo.TomoPlan(cfg, slope_model=tomo.TOMO_FFTMODEL)
    s2, var = pl.noise()
    assert abs(var / osys.slope_var - 1) < 5e-3
    s = f32(data["slopes"][0].ravel())
    d_o = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
    pl.apply_css(dev(s), d_o)
    torch.cuda.synchronize()
    assert rel(d_o.cpu().numpy(), osys.apply_A(s)) <= 1e-2
    _, h = osys.solve_cg(s, 1000)
    n_it = int(np.flatnonzero(h / h[0] < 1e-6)[0])
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    e = rel(d_w.cpu().numpy().reshape(len(cfg.targets), -1)[0], osys.reconstruct(osys.solve_direct(s), 0))
    print(f"[FFT model, builder's generators] converged wavefront vs the continuous-integral oracle: {e:.2e}")
    assert e <= 1e-2
    pl.close()


ALL = ["cfg1", "small_lgs", "small_odd_focus", "small_fried", "small_fftmodel", "ngs_offaxis", "cfg2"]
# both solvers go through every solve gate: the multi-kernel CUDA-graph loop and the persistent cooperative kernel
SOLVERS = [tomo.TOMO_SOLVER_MULTIKERNEL, tomo.TOMO_SOLVER_PERSISTENT]
solvers = pytest.mark.parametrize("solver", SOLVERS, ids=["multikernel", "persistent"])


# ------------------------------------------------------------------------------------------------ P-a
@solvers
@pytest.mark.parametrize("name", ALL)
def test_mvm_parity(name, solver):
    """tomo_apply_css = the product of the plan's solver: one single-product launch of k_persistent, or k_rows_fwd / k_cols /
    k_rows_inv of the multi-kernel solver."""
    cfg, _, osys, data = system(name)
    pl = make_plan(name, solver=solver)
    cases = {"white": screens.random_vector(cfg, osys.Ns), "slopes": data["slopes"][0].ravel(),
             "cg_iterate": osys.solve_cg(data["slopes"][0].ravel(), 7)[0]}
    for label, v in cases.items():
        d_v, d_o = dev(v), torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
        pl.apply_css(d_v, d_o)
        torch.cuda.synchronize()
        assert_close(d_o.cpu().numpy(), osys.apply_A(f32(v)), TOL_MVM, what=(name, label))
    pl.close()


@pytest.mark.parametrize("name", ALL)
def test_target_projection_parity(name):
    cfg, _, osys, data = system(name)
    pl = make_plan(name)
    zeta = osys.solve_cg(data["slopes"][0].ravel(), cfg.n_iter)[0]
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.apply_cos(dev(zeta), d_w)
    torch.cuda.synchronize()
    got = d_w.cpu().numpy().reshape(len(cfg.targets), -1)
    for t in range(len(cfg.targets)):
        assert_close(got[t], osys.reconstruct(f32(zeta), t), TOL_MVM, what=(name, t))
    pl.close()


# ------------------------------------------------------------------------------------------------ P-b
@solvers
@pytest.mark.parametrize("name", ["cfg1", "small_lgs", "small_odd_focus", "ngs_offaxis", "cfg2"])
def test_teacher_forced_cg_steps(name, solver):
    cfg, _, osys, data = system(name)
    pl = make_plan(name, solver=solver)
    n_it = cfg.n_iter
    _, _, st = osys.solve_cg(f32(data["slopes"][0].ravel()), n_it, record=True)
    ks = range(n_it) if osys.Ns < 1000 else range(0, n_it, 3)
    for k in ks:
        d_x, d_r, d_p = dev(st[k]["x"]), dev(st[k]["r"]), dev(st[k]["p"])
        sc = dev([st[k]["rho"], 0.0, 0.0], torch.float64)
        pl.cg_step(d_x, d_r, d_p, sc)
        torch.cuda.synchronize()
        nx = st[k + 1]
        # the oracle state was rounded to fp32 on upload: compare against a step taken from the rounded state
        if np.linalg.norm(nx["x"]) > 0:
            assert_close(d_x.cpu().numpy(), nx["x"], TOL_STEP, what=(name, k, "x"))
        assert_close(d_r.cpu().numpy(), nx["r"], TOL_STEP, what=(name, k, "r"))
        assert_close(d_p.cpu().numpy(), nx["p"], TOL_STEP, what=(name, k, "p"))
        rho1, alpha, beta = sc.cpu().numpy()
        assert abs(alpha / st[k]["alpha"] - 1) <= TOL_STEP and abs(beta / st[k]["beta"] - 1) <= TOL_STEP, (name, k)
        assert abs(rho1 / nx["rho"] - 1) <= TOL_STEP
    pl.close()


# ------------------------------------------------------------------------------------------------ P-c
def _horizon(h_a, h_b, x_a=None, x_b=None, tol=TOL_TRAJ):
    d = np.abs(h_a / h_b - 1.0)
    bad = np.flatnonzero(d > tol)
    return int(bad[0]) if bad.size else len(h_a)


@solvers
@pytest.mark.parametrize("name", ["cfg1", "small_lgs", "cfg2"])
def test_free_running_fp32_tracks_oracle_up_to_the_fp32_horizon(name, solver):
    cfg, _, osys, data = system(name)
    n_it = cfg.n_iter
    s = f32(data["slopes"][0].ravel())
    x64, h64 = osys.solve_cg(s, n_it)
    _, h32 = osys.solve_cg(s, n_it, dtype=np.float32)           # fp32 CPU emulation of the same algorithm
    k_star = max(_horizon(h32, h64) - 2, 3)
    pl = make_plan(name, solver=solver)
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    hg = pl.residuals(1, n_it)[0]
    d = np.abs(hg / h64 - 1.0)
    assert d[:k_star + 1].max() <= TOL_TRAJ, (name, k_star, d[:k_star + 1].max())
    # x_k up to the horizon: rerun with exactly k_star iterations (fixed-count solves are deterministic)
    pl.solve(dev(s), d_w, k_star)
    z = torch.empty(pl.slopes_len, dtype=torch.float32, device="cuda")
    pl.get_zeta(z)
    torch.cuda.synchronize()
    xk = osys.solve_cg(s, k_star)[0]
    assert_close(z.cpu().numpy(), xk, TOL_TRAJ, what=(name, k_star))
    print(f"[P-c {name}] fp32 horizon k*={k_star}; deviation of ||r_k|| at the full count {n_it}: {d[-1]:.2e}")
    pl.close()


# ------------------------------------------------------------------------------------------------ P-d
@solvers
@pytest.mark.parametrize("name", ["cfg1", "small_lgs", "small_odd_focus", "small_fried", "small_fftmodel", "ngs_offaxis", "cfg2"])
def test_converged_solution_matches_direct_solve(name, solver):
    cfg, _, osys, data = system(name)
    s = f32(data["slopes"][0].ravel())
    zeta = osys.solve_direct(s)
    # iterations until the ORACLE's CG reaches 1e-6 relative residual
    _, h = osys.solve_cg(s, 1000)
    n_it = int(np.flatnonzero(h / h[0] < 1e-6)[0])
    assert n_it <= 1000
    pl = make_plan(name, solver=solver)
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    got = d_w.cpu().numpy().reshape(len(cfg.targets), -1)
    for t in range(len(cfg.targets)):
        assert_close(got[t], osys.reconstruct(zeta, t), 1e-3, what=(name, t, n_it))
    pl.close()


# ------------------------------------------------------------------------------------------------ P-e
@pytest.mark.parametrize("name,prec", [("cfg1", tomo.TOMO_F64), ("small_lgs", tomo.TOMO_F64), ("cfg2", tomo.TOMO_F64),
                                        ("cfg1", tomo.TOMO_F32S_F64A)])
@solvers
def test_fp64_instantiation_meets_the_literal_gate_where_the_oracle_is_reproducible(name, prec, solver):
    cfg, _, osys, data = system(name)
    n_it = cfg.n_iter
    s = f32(data["slopes"][0].ravel())
    x_a, h_a = osys.solve_cg(s, n_it)
    # second fp64 oracle run differing only in rounding (rhs perturbed by 1e-15 relative)
    x_b, h_b = osys.solve_cg(s * (1.0 + 1e-15 * np.cos(np.arange(s.size))), n_it)
    k_rep = _horizon(h_b, h_a, tol=1e-4)
    phi_a, phi_b = osys.reconstruct(x_a, 0), osys.reconstruct(x_b, 0)
    reproducible = k_rep > n_it and rel(phi_b, phi_a) <= 1e-4
    pl = make_plan(name, precision=prec, solver=solver)
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    n_gate = n_it
    if not reproducible:
        # the wavefront is 10-1000x more sensitive than the residual history (C_os amplifies the low-order content):
        # the reproducibility horizon is where BOTH still agree between the two oracle runs, minus 2
        n_gate = max(min(k_rep, n_it), 3)
        while n_gate > 3:
            xa_k, xb_k = osys.solve_cg(s, n_gate)[0], osys.solve_cg(s * (1.0 + 1e-15 * np.cos(np.arange(s.size))), n_gate)[0]
            if rel(osys.reconstruct(xb_k, 0), osys.reconstruct(xa_k, 0)) <= 1e-4:
                break
            n_gate -= 1
        n_gate = max(n_gate - 2, 3)
    pl.solve(dev(s), d_w, n_gate)
    torch.cuda.synchronize()
    hg = pl.residuals(1, n_gate)[0]
    xo, ho = osys.solve_cg(s, n_gate)
    tol_h = TOL_TRAJ
    assert np.abs(hg / ho - 1.0).max() <= tol_h, (name, n_gate, np.abs(hg / ho - 1.0).max())
    e = rel(d_w.cpu().numpy().reshape(len(cfg.targets), -1)[0], osys.reconstruct(xo, 0))
    if prec == tomo.TOMO_F64:
        assert e <= TOL_TRAJ, (name, n_gate, e)
    print(f"[P-e {name} prec={prec}] oracle reproducible to k={k_rep}; gated at {n_gate} iterations: wavefront {e:.2e}")
    pl.close()


# ------------------------------------------------------------------------------------------------ API behaviour
@solvers
def test_batch_frames_equal_single_solves_bitwise_and_residuals(solver):
    cfg, _, osys, data = system("small_lgs")
    pl = make_plan("small_lgs", max_batch=2, solver=solver)
    s = data["slopes"].reshape(2, -1)
    n_it = 12
    d_w2 = torch.empty(2 * pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve_batch(dev(s), d_w2, 2, n_it)
    torch.cuda.synchronize()
    h2 = pl.residuals(2, n_it)
    for f in range(2):
        d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
        pl.solve(dev(s[f]), d_w, n_it)
        torch.cuda.synchronize()
        assert torch.equal(d_w, d_w2[f * pl.wavefront_len:(f + 1) * pl.wavefront_len])
        assert np.array_equal(pl.residuals(1, n_it)[0], h2[f])
    pl.close()


@solvers
def test_zero_iterations_and_warm_start(solver):
    cfg, _, osys, data = system("small_lgs")
    pl = make_plan("small_lgs", solver=solver)
    s = f32(data["slopes"][0].ravel())
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, 0)                                   # x = 0 -> phi = 0, history = [||M s||]
    torch.cuda.synchronize()
    assert float(d_w.abs().max()) == 0.0
    assert abs(pl.residuals(1, 0)[0, 0] / np.linalg.norm(osys.rhs(s)) - 1) < 1e-6
    # warm start: from the oracle's 6-iteration iterate, 5 more iterations
    x6 = osys.solve_cg(s, 6)[0]
    xo, ho = osys.solve_cg(s, 5, x0=f32(x6))
    pl.solve_batch(dev(s), d_w, 1, 5, x0=dev(x6))
    z = torch.empty(pl.slopes_len, dtype=torch.float32, device="cuda")
    pl.get_zeta(z)
    torch.cuda.synchronize()
    assert np.abs(pl.residuals(1, 5)[0] / ho - 1).max() <= TOL_TRAJ
    assert_close(z.cpu().numpy(), xo, TOL_TRAJ, what="warm start")
    pl.close()


def test_caller_supplied_generators_and_not_ready():
    cfg, _, osys, data = system("cfg1")
    pl = tomo.TomoPlan(cfg, upload=False)
    d_v = dev(data["slopes"][0].ravel())
    with pytest.raises(tomo.TomoError) as e:
        pl.apply_css(d_v, torch.empty_like(d_v))
    assert e.value.code == tomo.TOMO_ENOTREADY
    gen = 2.0 * tomo.host_css_generators(cfg)                  # doubled covariance: A v = 2 C v + sigma^2 v
    pl.upload_kernels(css_gen=gen)
    d_o = torch.empty_like(d_v)
    pl.apply_css(d_v, d_o)
    torch.cuda.synchronize()
    v = f32(data["slopes"][0].ravel())
    ref = 2.0 * osys.css_unprojected(v) + osys.sigma2 * v
    assert_close(d_o.cpu().numpy(), ref, TOL_MVM, what="doubled generators")
    pl.close()


def test_persistent_solver_falls_back_to_the_multikernel_solver_for_other_fft_edges():
    """n = 25 pads to P = 50 = 2 * 5^2, an edge the persistent kernel is not instantiated for: the default solver must hand
    over to the multi-kernel path (include/tomo.h) and still meet the gates."""
    cfg = small_lgs_config(n=25, n_gs=3, n_layers=3, targets=((0.0, 0.0),))
    osys = OracleSystem(cfg)
    data = screens.generate(cfg, osys.sigma2, n_frames=1)
    s = f32(data["slopes"][0].ravel())
    pl = tomo.TomoPlan(cfg)                     # default: persistent
    assert pl.P == 50
    used, note = pl.solver_in_use()             # decided at upload, reported, never changed inside a solve
    assert used == tomo.TOMO_SOLVER_MULTIKERNEL and "FFT edge" in note, (used, note)
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    n_it = 8
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    assert pl.stats()["launches_last_solve"] > 4 * n_it          # one launch per phase, not one per solve
    x_or, h_or = osys.solve_cg(s, n_it)
    assert np.abs(pl.residuals(1, n_it)[0] / h_or - 1.0).max() <= TOL_TRAJ
    d_z = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
    pl.get_zeta(d_z)
    torch.cuda.synchronize()
    assert_close(d_z.cpu().numpy(), x_or, TOL_TRAJ, what="zeta_8")
    # the wavefront of an unconverged iterate amplifies the low-order content of the zeta deviation:
    # the projection is gated on the oracle's iterate
    pl.apply_cos(dev(x_or), d_w)
    torch.cuda.synchronize()
    assert_close(d_w.cpu().numpy(), osys.reconstruct(f32(x_or), 0), TOL_MVM, what="C_os zeta")
    pl.close()
