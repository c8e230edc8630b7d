"""Parity at BASELINE.json's full sizes of the kernel bench.py times: every call below goes through a plan whose solver is
the persistent one (asserted with tomo_get_solver), so tomo_apply_css is ONE single-product launch of k_persistent,
tomo_cg_step one teacher-forced iteration of it and tomo_solve the whole solve; the test ids name the instantiation
(FFT edge P, channel count C = 2 n_wfs) they exercise:

    cfg3   k_persistent<P=160>, C=12      cfg4   k_persistent<P=160>, C=16 (10 targets)
    cfg5   n = 16, 32, 64, 96, 128  ->  k_persistent<P=32, 64, 128, 192, 256>, C=12

The dense oracle does not fit at ELT scale (51 648^2 fp64 = 21 GB; the 35-layer dense build already takes 5 minutes at
n = 16), so:
  * sampled outputs: rows of W Sigma_ss W^T the oracle builds one by one from subaperture POSITIONS
    (OracleSystem.css_rows_explicit: no generators, no Toeplitz indexing, no FFT); tip/tilt removal only shifts a
    channel by a constant, so the difference of two outputs of the same channel is compared;
  * every output: the matrix-free direct-sum oracle (oracle/directsum.c: entry by entry from the generators, no FFT) for
    the whole product, teacher-forced CG steps (P-b) from the oracle's own states, free-running iterations below the
    fp32 horizon, the literal full-count gate in fp64 (P-e) and the target projection (oracle cos_matrix_free).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.system import OracleSystem  # noqa: E402
from paper_1806_07938_b200 import tomo  # noqa: E402
from tomo_inputs import screens  # noqa: E402
from tomo_inputs.configs import get_config  # noqa: E402

from gates import assert_close, rel  # noqa: E402

pytestmark = pytest.mark.gpu


def dev(a, dtype=torch.float32):
    return torch.tensor(np.ascontiguousarray(a), dtype=dtype, device="cuda")


def f32(a):
    return np.asarray(a, dtype=np.float32).astype(np.float64)


def _gen_rows(args):
    from oracle import toeplitz as tz
    (n, d, dirs, h_gs, h, frac, r0, L0, model, i) = args
    return tz.css_generators(n, d, dirs, h_gs, h, frac, r0, L0, model, wfs_rows=[i])


def _build_generators_in_parallel(osys):
    """The oracle's generator table, unchanged arithmetic (oracle.toeplitz.css_generators), one process per output WFS:
    single-threaded it takes ~200 s at cfg3."""
    from concurrent.futures import ProcessPoolExecutor
    c = osys.cfg
    jobs = [(osys.n, osys.d, osys.dirs, osys.h_gs, list(c.h), list(c.frac), c.r0, c.L0, osys.model, i) for i in range(osys.N)]
    with ProcessPoolExecutor(max_workers=osys.N) as ex:
        osys.theta = sum(ex.map(_gen_rows, jobs))


_sys = {}


def matrix_free_system(name, build_cos=True):
    """(cfg, matrix-free oracle with its generator table, slopes of frame 0), built once per test session."""
    if name not in _sys:
        cfg = get_config(name)
        osys = OracleSystem(cfg, dense=False, build_cos=build_cos)
        _build_generators_in_parallel(osys)
        s = f32(screens.generate(cfg, osys.sigma2, n_frames=1)["slopes"][0].ravel())
        _sys[name] = (cfg, osys, s)
    return _sys[name]


def persistent_plan(cfg, osys=None, **kw):
    pl = tomo.TomoPlan(cfg, solver=tomo.TOMO_SOLVER_PERSISTENT, **kw)
    used, note = pl.solver_in_use()
    assert used == tomo.TOMO_SOLVER_PERSISTENT, note          # the kernel under test is k_persistent, not the fallback
    if osys is not None:
        assert pl.n_vs == osys.nv and abs(pl.noise()[0][0] / osys.sigma2 - 1) < 1e-12
    return pl


def apply_css(pl, v):
    d_o = torch.empty(pl.slopes_len, dtype=torch.float32, device="cuda")
    pl.apply_css(dev(v), d_o)
    torch.cuda.synchronize()
    assert pl.stats()["launches_last_solve"] <= 2             # one k_persistent launch + the fp32 conversion
    return d_o.cpu().numpy().astype(np.float64)


def teacher_forced_steps(pl, osys, s, ks, n_record):
    """P-b through tomo_cg_step (one PM_STATE launch of k_persistent) from the matrix-free oracle's states."""
    _, _, st = osys.solve_cg(s, n_record, record=True)
    worst = 0.0
    for k in ks:
        d_x, d_r, d_p = dev(st[k]["x"]), dev(st[k]["r"]), dev(st[k]["p"])
        sc = dev([st[k]["rho"], 0.0, 0.0], torch.float64)
        pl.cg_step(d_x, d_r, d_p, sc)
        torch.cuda.synchronize()
        nx = st[k + 1]
        if np.linalg.norm(nx["x"]) > 0:
            worst = max(worst, assert_close(d_x.cpu().numpy(), nx["x"], 1e-4, what=("x", k))[1])
        worst = max(worst, assert_close(d_r.cpu().numpy(), nx["r"], 1e-4, what=("r", k))[1])
        worst = max(worst, assert_close(d_p.cpu().numpy(), nx["p"], 1e-4, what=("p", k))[1])
        rho1, alpha, beta = sc.cpu().numpy()
        assert abs(alpha / st[k]["alpha"] - 1) <= 1e-4 and abs(beta / st[k]["beta"] - 1) <= 1e-4, (k, alpha, beta)
        assert abs(rho1 / nx["rho"] - 1) <= 1e-4
    return worst


# ------------------------------------------------------------------------------------------------ sampled outputs from positions
def _sampled_pairs_check(name, n_pairs, seed):
    """A v through k_persistent vs explicit rows of W Sigma_ss W^T: (A v)[r1] - (A v)[r2] for r1, r2 in the same channel."""
    cfg = get_config(name)
    osys = OracleSystem(cfg, dense=False, build_cos=False)
    pl = persistent_plan(cfg, osys, build_cos=False)
    v = f32(screens.generate(cfg, osys.sigma2, n_frames=1)["slopes"][0].ravel())
    got = apply_css(pl, v)
    u = osys.project_slopes(v)
    rng = np.random.default_rng(seed)
    worst = 0.0
    scale = float(np.sqrt(np.mean(got ** 2)))
    for _ in range(n_pairs):
        ch = int(rng.integers(0, 2 * osys.N))
        q1, q2 = (int(t) for t in rng.choice(osys.nv, size=2, replace=False))
        rows = [ch * osys.nv + q1, ch * osys.nv + q2]
        R = osys.css_rows_explicit(rows)
        want = (R[0] @ u + osys.sigma2 * u[rows[0]]) - (R[1] @ u + osys.sigma2 * u[rows[1]])
        have = got[rows[0]] - got[rows[1]]
        worst = max(worst, abs(have - want) / scale)
    pl.close()
    return worst


@pytest.mark.parametrize("name,n_pairs", [("cfg3", 4), ("cfg4", 3), ("cfg5_n16", 4), ("cfg5_n32", 3), ("cfg5_n64", 2),
                                          ("cfg5_n96", 2), ("cfg5_n128", 2)],
                         ids=["cfg3-P160-C12", "cfg4-P160-C16", "n16-P32", "n32-P64", "n64-P128", "n96-P192", "n128-P256"])
def test_persistent_product_on_sampled_outputs_from_positions(name, n_pairs):
    assert _sampled_pairs_check(name, n_pairs, seed=len(name) + n_pairs) <= 1e-5


# ------------------------------------------------------------------------------------------------ the sweep instances, every output
@pytest.mark.parametrize("n", [16, 32, 64, 96, 128], ids=["n16-P32", "n32-P64", "n64-P128", "n96-P192", "n128-P256"])
def test_sweep_persistent_product_and_teacher_forced_steps_against_the_matrix_free_oracle(n):
    cfg, osys, s = matrix_free_system(f"cfg5_n{n}", build_cos=False)
    pl = persistent_plan(cfg, osys, build_cos=False)
    assert pl.P == 2 * n
    e = assert_close(apply_css(pl, s), osys.apply_A(s), 1e-4, what=("A s", n))
    w = teacher_forced_steps(pl, osys, s, ks=(0, 1, 2), n_record=3)
    print(f"[sweep n={n} P={pl.P}] product rel-L2 {e[0]:.2e} max-abs/rms {e[1]:.2e}; teacher-forced steps max-abs/rms {w:.2e}")
    pl.close()
    _sys.pop(f"cfg5_n{n}", None)


# ------------------------------------------------------------------------------------------------ cfg3
def test_cfg3_persistent_product_steps_solve_and_projection_against_the_matrix_free_oracle():
    """Whole product, teacher-forced steps (P-b at n = 74), 12 free-running CG and MINRES iterations (below the fp32
    horizon) and the projection at cfg3."""
    cfg, osys, s = matrix_free_system("cfg3")
    pl = persistent_plan(cfg, osys)
    # P-a, every output
    assert_close(apply_css(pl, s), osys.apply_A(s), 1e-4, what="A s")
    # P-b: teacher-forced steps from the oracle's states
    teacher_forced_steps(pl, osys, s, ks=(0, 1, 2, 5, 8, 11), n_record=12)
    # P-c, free-running below the horizon
    n_it = 12
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    assert pl.stats()["launches_last_solve"] < n_it             # one launch per solve + the projection kernels
    x_or, h_or = osys.solve_cg(s, n_it)
    h_gpu = pl.residuals(1, n_it)[0]
    assert np.abs(h_gpu / h_or - 1.0).max() <= 1e-3
    d_z = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
    pl.get_zeta(d_z)
    torch.cuda.synchronize()
    assert_close(d_z.cpu().numpy(), x_or, 1e-3, what="zeta_12")
    # P-a for the projection alone (A7-A8) on the oracle's iterate
    pl.apply_cos(dev(x_or), d_w)
    torch.cuda.synchronize()
    assert_close(d_w.cpu().numpy(), osys.reconstruct(f32(x_or), 0), 1e-4, what="C_os zeta")
    # M-c at full size: 12 free-running MINRES iterations (tomo_solve_minres) against the oracle's MINRES on the same
    # matrix-free operator; the residual never increases and stays below CG's
    pl.solve_minres(dev(s), d_w, 1, n_it)
    pl.get_zeta(d_z)
    torch.cuda.synchronize()
    xm_or, hm_or = osys.solve_minres(s, n_it)
    hm_gpu = pl.residuals(1, n_it)[0]
    assert np.abs(hm_gpu / hm_or - 1.0).max() <= 1e-3
    assert_close(d_z.cpu().numpy(), xm_or, 1e-3, what="minres zeta_12")
    assert np.all(np.diff(hm_gpu) <= 0) and np.all(hm_gpu <= h_gpu * (1 + 1e-5))
    pl.close()


def test_cfg3_fp64_instantiation_meets_the_literal_gate_at_the_full_count():
    """P-e at ELT size: north_star's literal gate -- the fp64 instantiation of the same kernels (TOMO_F64), the config's 50
    iterations, residual history and wavefront within 1e-3 of the matrix-free fp64 oracle (two fp64 oracle runs agree
    with each other at cfg3 after 50 iterations; checked here on the history)."""
    cfg, osys, s = matrix_free_system("cfg3")
    n_it = cfg.n_iter
    assert n_it == 50
    x_a, h_a = osys.solve_cg(s, n_it)
    x_b, h_b = osys.solve_cg(s * (1.0 + 1e-15 * np.cos(np.arange(s.size))), n_it)
    assert np.abs(h_b / h_a - 1.0).max() <= 1e-4 and rel(x_b, x_a) <= 1e-4        # the oracle is reproducible at this count
    pl = persistent_plan(cfg, osys, precision=tomo.TOMO_F64)
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    h_gpu = pl.residuals(1, n_it)[0]
    dh = float(np.abs(h_gpu / h_a - 1.0).max())
    assert dh <= 1e-3, dh
    d_z = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
    pl.get_zeta(d_z)
    torch.cuda.synchronize()
    ez = assert_close(d_z.cpu().numpy(), x_a, 1e-3, what="zeta_50")
    ew = assert_close(d_w.cpu().numpy(), osys.reconstruct(x_a, 0), 1e-3, what="wavefront_50")
    print(f"[P-e cfg3 TOMO_F64, 50 iterations] history {dh:.2e}, zeta rel-L2 {ez[0]:.2e}, wavefront rel-L2 {ew[0]:.2e} max-abs/rms {ew[1]:.2e}")
    pl.close()


# ------------------------------------------------------------------------------------------------ cfg4
def test_cfg4_persistent_product_steps_and_moao_projection_against_the_matrix_free_oracle():
    """cfg4 (8 LGS on 120", C = 16, 10 targets): whole product, 8 teacher-forced steps from the matrix-free oracle's
    states, and the projection (k_cos_mac_inv streaming 734 MB of spectra) for targets 0 and 9 against the oracle's
    cos_matrix_free (Eq.32 entry by entry, no FFT)."""
    cfg, osys, s = matrix_free_system("cfg4")
    pl = persistent_plan(cfg, osys)
    assert_close(apply_css(pl, s), osys.apply_A(s), 1e-4, what="A s")
    teacher_forced_steps(pl, osys, s, ks=range(8), n_record=8)
    x_or = osys.solve_cg(s, 8)[0]
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.apply_cos(dev(x_or), d_w)
    torch.cuda.synchronize()
    got = d_w.cpu().numpy().reshape(len(cfg.targets), -1)
    for t in (0, 9):
        assert_close(got[t], osys.reconstruct(f32(x_or), t), 1e-4, what=("C_os zeta, target", t))
    pl.close()
    _sys.pop("cfg4", None)


# ------------------------------------------------------------------------------------------------ batch instance
@pytest.mark.parametrize("name,frames", [("cfg3", (3, 5)), ("cfg4", (3,)), ("cfg5_n128", (2,)), ("cfg5_n128", (16,))],
                         ids=["cfg3-P160-C12", "cfg4-P160-C16", "n128-P256", "n128-P256-b16-one-frame-per-pass"])
def test_batch_instance_equals_single_solves_bitwise(name, frames):
    """Batch path at full size: with several frames the slab passes are balanced over the CTAs and some spectra are read
    through L2 instead of shared memory.  Same arithmetic in the same order, so every frame must equal its single-frame
    solve bit for bit (zeta, residual history, wavefront) -- which ties the batch instance to the single-frame one the
    tests above compare with the oracle."""
    cfg = get_config(name)
    B, n_it = max(frames), 6
    pl = persistent_plan(cfg, max_batch=B)
    data = screens.generate(cfg, float(pl.noise()[0][0]), n_frames=B)
    s = np.ascontiguousarray(data["slopes"].reshape(B, -1), dtype=np.float32)
    singles = []
    for f in range(B):
        d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
        d_z = torch.empty(pl.slopes_len, dtype=torch.float32, device="cuda")
        pl.solve(dev(s[f]), d_w, n_it)
        pl.get_zeta(d_z)
        torch.cuda.synchronize()
        singles.append((d_w.clone(), d_z.clone(), pl.residuals(1, n_it)[0].copy()))
    for nb in frames:
        d_w = torch.empty(nb * pl.wavefront_len, dtype=torch.float32, device="cuda")
        d_z = torch.empty(nb * pl.slopes_len, dtype=torch.float32, device="cuda")
        pl.solve_batch(dev(s[:nb]), d_w, nb, n_it)
        pl.get_zeta(d_z, nb)
        torch.cuda.synchronize()
        h = pl.residuals(nb, n_it)
        for f in range(nb):
            assert torch.equal(d_w[f * pl.wavefront_len:(f + 1) * pl.wavefront_len], singles[f][0]), (nb, f)
            assert torch.equal(d_z[f * pl.slopes_len:(f + 1) * pl.slopes_len], singles[f][1]), (nb, f)
            assert np.array_equal(h[f], singles[f][2]), (nb, f)
    pl.close()
