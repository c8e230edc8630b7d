"""Layered-phase (MCAO) plans, tomo_options.layered (PAPER.md S2.D L199, S6 L516; reading G31): parity of the CUDA path with
oracle/layered.py (dense, from positions) at small sizes and with the oracle's entry-by-entry direct sum at ELT size.

Gates: rel-L2 <= 1e-4 as for the LTAO projection (P-a); max-abs <= 3e-5 of the rms of the expected layer: the element error
of the fp32 path scales with the largest values of the grid (measured 1.0e-5 rms), and the rms over a meta-pupil grid -- most
of it outside the guide-star footprints, where the estimate falls to zero -- is a few times smaller than over a pupil."""
from dataclasses import replace

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import directsum  # noqa: E402
from oracle import layered as lay  # noqa: E402
from oracle import toeplitz as tz  # noqa: E402
from oracle.system import OracleSystem  # noqa: E402
from paper_1806_07938_b200 import tomo  # noqa: E402
from tomo_inputs import screens  # noqa: E402
from tomo_inputs.configs import get_config, small_lgs_config  # noqa: E402

from gates import assert_close  # noqa: E402

pytestmark = pytest.mark.gpu

TOL = 1e-4
TOL_MAX = 3e-5


def dev(a):
    return torch.tensor(np.ascontiguousarray(a), dtype=torch.float32, device="cuda")


def f32(a):
    return np.asarray(a, dtype=np.float32).astype(np.float64)


CASES = {
    "ngs": (lambda: replace(get_config("cfg1"), h=(0.0, 4000.0, 11000.0), frac=(0.55, 0.25, 0.2)), 30.0, "hudgin"),
    "lgs": (lambda: small_lgs_config(n=10, n_gs=3, n_layers=3), 20.0, "hudgin"),
    "lgs_odd_focus_fried": (lambda: replace(small_lgs_config(n=11, n_gs=3, n_layers=2, n_remove=3), obstruction=0.3), 45.0, "fried"),
}
_cache = {}


def system(name):
    if name not in _cache:
        mk, fov, model = CASES[name]
        cfg = mk()
        osys = OracleSystem(cfg, model=model, build_cos=False)
        _cache[name] = (cfg, fov, model, osys, screens.generate(cfg, osys.sigma2, n_frames=3))
    return _cache[name]


def oracle_layers(name, zeta):
    cfg, fov, model, osys, _ = system(name)
    n_m = lay.n_meta(cfg.n, cfg.d, cfg.h, osys.h_gs, fov)
    z = osys.project_slopes(zeta)                                   # W_s^T M_s^T zeta (M_s symmetric, Eq.36)
    return n_m, lay.layered_estimate(z, n_m, osys.centres, cfg.d, osys.dirs, osys.h_gs, cfg.h, cfg.frac, cfg.r0, cfg.L0, model)


def plan(name, **kw):
    cfg, fov, model, osys, _ = system(name)
    sm = {"fried": tomo.TOMO_FRIED}.get(model, tomo.TOMO_HUDGIN)
    pl = tomo.TomoPlan(cfg, slope_model=sm, layered=True, fov_radius=fov, **kw)
    assert pl.solver_in_use()[0] == kw.get("solver", tomo.TOMO_SOLVER_PERSISTENT), pl.solver_in_use()
    return pl


@pytest.mark.parametrize("name", list(CASES))
def test_layer_projection_parity(name):
    cfg, fov, _, osys, data = system(name)
    pl = plan(name)
    zeta = osys.solve_cg(data["slopes"][0].ravel(), 12)[0]
    n_m, want = oracle_layers(name, f32(zeta))
    assert pl.n_prime == n_m and pl.n_vphi == n_m * n_m and pl.wavefront_len == len(cfg.h) * n_m * n_m
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.apply_cos(dev(zeta), d_w)
    torch.cuda.synchronize()
    got = d_w.cpu().numpy().reshape(len(cfg.h), n_m, n_m)
    for k in range(len(cfg.h)):
        assert_close(got[k].ravel(), want[k].ravel(), TOL, TOL_MAX, what=(name, "layer", k))
    pl.close()


@pytest.mark.parametrize("solver", [tomo.TOMO_SOLVER_MULTIKERNEL, tomo.TOMO_SOLVER_PERSISTENT], ids=["multikernel", "persistent"])
@pytest.mark.parametrize("name", ["ngs", "lgs"])
def test_layered_solve_to_convergence_against_the_direct_solution(name, solver):
    """Whole path on a layered plan: CG to convergence, then every layer; against Sigma_{phi_k s} (direct solution)."""
    cfg, _, _, osys, data = system(name)
    pl = plan(name, solver=solver, max_batch=3)
    S = np.stack([data["slopes"][f].ravel() for f in range(3)])
    _, h = osys.solve_cg(S[0], 1000)
    n_it = int(np.flatnonzero(h / h[0] < 1e-6)[0])
    d_w = torch.empty(3 * pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve_batch(dev(S), d_w, 3, n_it)
    torch.cuda.synchronize()
    got = d_w.cpu().numpy().reshape(3, -1)
    for f in range(3):
        _, want = oracle_layers(name, osys.solve_direct(f32(S[f])))
        assert_close(got[f], want.ravel(), 1e-3, what=(name, "frame", f))
    # frames of a batch are bitwise the single solves; MINRES goes through the same projection
    d_1 = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(S[1]), d_1, n_it)
    torch.cuda.synchronize()
    assert np.array_equal(d_1.cpu().numpy(), got[1])
    pl.solve_minres(dev(S), d_w, 3, n_it)
    torch.cuda.synchronize()
    _, want = oracle_layers(name, osys.solve_direct(f32(S[2])))
    assert_close(d_w.cpu().numpy().reshape(3, -1)[2], want.ravel(), 1e-3, what=(name, "minres"))
    pl.close()


def test_ray_traced_layers_reproduce_the_ltao_plan_on_a_grid_aligned_direction():
    """NGS: a target whose footprint shift h_k beta is a whole number of grid steps in every layer.  The layered plan's
    output, ray-traced (pure selection), must equal the LTAO plan's Sigma_{phi_beta s} product before M_phi (piston removed
    from both here) -- two different plans of the library against each other and against the oracle."""
    base = replace(get_config("cfg1"), h=(0.0, 5000.0, 10000.0), frac=(0.5, 0.3, 0.2))
    step = base.d / 5000.0 / (np.pi / 180 / 3600)
    cfg = replace(base, targets=((2 * step, -1 * step),))
    osys = OracleSystem(cfg)
    zeta = osys.solve_cg(screens.generate(cfg, osys.sigma2, n_frames=1)["slopes"][0].ravel(), 10)[0]
    p_l = tomo.TomoPlan(cfg, layered=True, fov_radius=4.5 * step)
    p_t = tomo.TomoPlan(cfg)
    d_l = torch.empty(p_l.wavefront_len, dtype=torch.float32, device="cuda")
    d_t = torch.empty(p_t.wavefront_len, dtype=torch.float32, device="cuda")
    p_l.apply_cos(dev(zeta), d_l)
    p_t.apply_cos(dev(zeta), d_t)
    torch.cuda.synchronize()
    n_m = p_l.n_prime
    layers = d_l.cpu().numpy().astype(np.float64).reshape(3, n_m, n_m)
    traced = lay.ray_trace(layers, osys.phase_pts, cfg.d, osys.h_gs, cfg.h, cfg.targets[0])
    traced -= traced.mean()                                     # M_phi of an NGS system removes piston only (G14)
    assert_close(traced, d_t.cpu().numpy().astype(np.float64), 1e-4, tol_max=2e-5, what="layered vs LTAO plan")
    assert_close(traced, osys.reconstruct(f32(zeta), 0), 1e-4, tol_max=2e-5, what="layered vs oracle LTAO")
    p_l.close()
    p_t.close()


def test_layered_plan_at_elt_size_against_the_direct_sum():
    """cfg3 geometry (n = 74, 6 LGS, P = 160) as an MCAO system with a 60 arcsec field radius: every layer grid of the
    product through k_cos_* against the oracle's entry-by-entry sum over the generators xi'_k (no FFT), all outputs."""
    cfg = get_config("cfg3")
    osys = OracleSystem(cfg, dense=False, build_cos=False)
    fov = 60.0
    n_m = lay.n_meta(cfg.n, cfg.d, cfg.h, osys.h_gs, fov)
    pl = tomo.TomoPlan(cfg, layered=True, fov_radius=fov)
    assert pl.n_prime == n_m and pl.solver_in_use()[0] == tomo.TOMO_SOLVER_PERSISTENT
    zeta = f32(screens.random_vector(cfg, osys.Ns))
    z = osys.project_slopes(zeta)
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.apply_cos(dev(zeta), d_w)
    torch.cuda.synchronize()
    got = d_w.cpu().numpy().reshape(len(cfg.h), n_m, n_m)
    worst = 0.0
    for k, (hk, fk) in enumerate(zip(cfg.h, cfg.frac)):
        xi = tz.cos_generators(cfg.n, n_m, cfg.d, osys.dirs, osys.h_gs, (0.0, 0.0), [hk], [fk], cfg.r0, cfg.L0)[0]
        want = directsum.cos_layer(xi, cfg.n, n_m, osys.ix, osys.iy, z)
        e2, em = assert_close(got[k].ravel(), want.ravel(), TOL, TOL_MAX, what=("cfg3 layered", k))
        worst = max(worst, e2)
    print(f"[layered cfg3, n_m = {n_m}, P_os = {pl.P_os}] worst layer rel-L2 {worst:.2e}")
    # a sampled set of grid points from POSITIONS (the generator route itself is pinned on CPU at small sizes)
    rng = np.random.default_rng(11)
    for k in (0, len(cfg.h) // 2, len(cfg.h) - 1):
        g = (osys.h_gs - cfg.h[k]) / osys.h_gs
        u = lay.layer_grid(n_m, g * cfg.d)
        pick = rng.choice(n_m * n_m, size=6, replace=False)
        from oracle.covariance import cov_phase_slope
        for m in pick:
            acc = 0.0
            for j in range(osys.N):
                pos = g * osys.centres + cfg.h[k] * np.asarray(osys.dirs[j]) * (np.pi / 180 / 3600)
                for b in range(2):
                    row = cfg.frac[k] * cov_phase_slope(pos - u[m][None, :], b, g * cfg.d, 1.0 / cfg.d, cfg.r0, cfg.L0)
                    acc += row @ z.reshape(osys.N, 2, osys.nv)[j, b]
            scale = np.sqrt(np.mean(got[k].astype(np.float64) ** 2))
            assert abs(got[k].ravel()[m] - acc) <= 1e-5 * scale + 1e-4 * abs(acc), (k, m, got[k].ravel()[m], acc)
    pl.close()


def test_layered_plan_rejects_targets_and_negative_field():
    import ctypes as C
    cfg = small_lgs_config(n=8, n_gs=3, n_layers=2)
    lib = tomo.load()
    pr = tomo._Problem(cfg)                                      # keeps cfg's targets
    opt = tomo._Options(0, 0, 0, 1, 0, tomo.TOMO_SOLVER_PERSISTENT, 1, 1, 10.0)
    h = C.c_void_p()
    noise = tomo._Noise(None, 0.1, None, None)
    assert lib.tomo_plan_create(pr.geom, pr.cn2, cfg.r0, cfg.L0, noise, opt, C.byref(h)) == tomo.TOMO_EINVAL
    with pytest.raises(tomo.TomoError):
        tomo.TomoPlan(cfg, layered=True, fov_radius=-1.0)
