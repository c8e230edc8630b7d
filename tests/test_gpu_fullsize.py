"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (persistent solver, fp32, batch 1).

The dense oracle does not fit at ELT scale (51 648^2 fp64 = 21 GB), so:
  * the product is checked on SAMPLED outputs the oracle computes one by one from subaperture POSITIONS
    (OracleSystem.css_rows_explicit: no generators, no Toeplitz indexing, no FFT): tip/tilt removal only shifts a
    channel by a constant, so the difference of two outputs of the same channel is compared;
  * cfg3 additionally runs the matrix-free direct-sum oracle (oracle/directsum.c) for the whole product, a fixed number
    of CG iterations below the fp32 horizon (~35 at cfg3) and the target projection.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.system import OracleSystem  # noqa: E402
from paper_1806_07938_b200 import tomo  # noqa: E402
from tomo_inputs import screens  # noqa: E402
from tomo_inputs.configs import get_config  # noqa: E402

pytestmark = pytest.mark.gpu


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def dev(a):
    return torch.tensor(np.ascontiguousarray(a), dtype=torch.float32, device="cuda")


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


def _sampled_pairs_check(name, n_pairs, seed):
    """A v on the GPU vs explicit rows of W Sigma_ss W^T: (A v)[r1] - (A v)[r2] for r1, r2 in the same channel."""
    cfg = get_config(name)
    osys = OracleSystem(cfg, dense=False, build_cos=False)
    pl = tomo.TomoPlan(cfg, solver=tomo.TOMO_SOLVER_PERSISTENT, build_cos=False)
    assert pl.n_vs == osys.nv and abs(pl.noise()[0][0] / osys.sigma2 - 1) < 1e-12
    data = screens.generate(cfg, osys.sigma2, n_frames=1)
    v = f32(data["slopes"][0].ravel())
    d_o = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
    pl.apply_css(dev(v), d_o)
    torch.cuda.synchronize()
    got = d_o.cpu().numpy().astype(np.float64)
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


def test_cfg3_product_on_sampled_outputs_from_positions():
    assert _sampled_pairs_check("cfg3", n_pairs=4, seed=3) <= 1e-4


def test_cfg4_product_on_sampled_outputs_from_positions():
    assert _sampled_pairs_check("cfg4", n_pairs=3, seed=4) <= 1e-4


@pytest.mark.parametrize("n", [64, 128])
def test_sweep_sizes_product_on_sampled_outputs_from_positions(n):
    assert _sampled_pairs_check(f"cfg5_n{n}", n_pairs=2, seed=n) <= 1e-4


def test_cfg3_solve_and_projection_against_the_matrix_free_oracle():
    """Whole product, 12 free-running CG and MINRES iterations (below the fp32 horizon) and the projection at cfg3."""
    cfg = get_config("cfg3")
    osys = OracleSystem(cfg, dense=False)
    _build_generators_in_parallel(osys)
    data = screens.generate(cfg, osys.sigma2, n_frames=1)
    s = f32(data["slopes"][0].ravel())
    pl = tomo.TomoPlan(cfg, solver=tomo.TOMO_SOLVER_PERSISTENT)
    # P-a, every output
    d_o = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
    pl.apply_css(dev(s), d_o)
    torch.cuda.synchronize()
    assert rel(d_o.cpu().numpy(), osys.apply_A(s)) <= 1e-4
    # P-c, free-running below the horizon
    n_it = 12
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    x_or, h_or = osys.solve_cg(s, n_it)
    h_gpu = pl.residuals(1, n_it)[0]
    assert np.abs(h_gpu / h_or - 1.0).max() <= 1e-3
    d_z = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
    pl.get_zeta(d_z)
    torch.cuda.synchronize()
    assert rel(d_z.cpu().numpy(), x_or) <= 1e-3
    # P-a for the projection alone (A7-A8) on the oracle's iterate
    pl.apply_cos(dev(x_or), d_w)
    torch.cuda.synchronize()
    assert rel(d_w.cpu().numpy(), osys.reconstruct(f32(x_or), 0)) <= 1e-4
    # M-c at full size: 12 free-running MINRES iterations (tomo_solve_minres) against the oracle's MINRES on the same
    # matrix-free operator; the residual never increases and stays below CG's
    pl.solve_minres(dev(s), d_w, 1, n_it)
    pl.get_zeta(d_z)
    torch.cuda.synchronize()
    xm_or, hm_or = osys.solve_minres(s, n_it)
    hm_gpu = pl.residuals(1, n_it)[0]
    assert np.abs(hm_gpu / hm_or - 1.0).max() <= 1e-3
    assert rel(d_z.cpu().numpy(), xm_or) <= 1e-3
    assert np.all(np.diff(hm_gpu) <= 0) and np.all(hm_gpu <= h_gpu * (1 + 1e-5))
    pl.close()


def test_cfg3_batch_with_helped_slabs_equals_single_solves_bitwise():
    """Batch path at ELT size: with 3 and 5 frames the k_x slabs that have a single CTA hand frames to CTAs of other slabs,
    which read the spectra through L2 instead of shared memory (persist_kernel.cuh, slab_segments).  Same arithmetic in the
    same order, so every frame must equal its single-frame solve bit for bit (zeta, residual history, wavefront)."""
    cfg = get_config("cfg3")
    B, n_it = 5, 6
    pl = tomo.TomoPlan(cfg, solver=tomo.TOMO_SOLVER_PERSISTENT, max_batch=B)
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
    for nb in (3, B):
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
