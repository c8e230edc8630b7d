"""2 x 2 block-diagonal noise covariance of elongated LGS spots (NEXT rank 3) through the C ABI
(tomo_noise.sigma_xy_subap) against the dense oracle with the same blocks: product (P-a), free-running solve up to the
fp32 horizon (P-c), converged solve vs the direct solution (P-d).  The default (persistent) solver hands over to the
multi-kernel solver for non-diagonal noise."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.system import OracleSystem  # noqa: E402
from paper_1806_07938_b200 import tomo  # noqa: E402
from tomo_inputs import screens  # noqa: E402
from tomo_inputs.configs import small_lgs_config  # noqa: E402
from test_gpu_parity import TOL_MVM, TOL_TRAJ, _horizon, dev, f32, rel  # noqa: E402

pytestmark = pytest.mark.gpu


def _setup(n=10, n_remove=2):
    cfg = small_lgs_config(n=n, n_gs=3, n_layers=3, n_remove=n_remove, targets=((4.0, -2.0),))
    base = OracleSystem(cfg, build_cos=False)
    blocks = screens.elongated_noise_blocks(cfg, base.sigma2, elongation=2.5)
    osys = OracleSystem(cfg, noise_blocks=blocks)
    data = screens.generate(cfg, base.sigma2)
    s = f32(screens.add_block_noise(cfg, data["slopes_noiseless"], blocks)[0].ravel())
    diag = np.stack([blocks[0], blocks[1]], axis=1)                      # [n_wfs][2][n_vs]
    pl = tomo.TomoPlan(cfg, sigma2_subap=diag, sigma_xy_subap=blocks[2])
    return cfg, osys, pl, s, blocks


@pytest.mark.parametrize("n,n_remove", [(10, 2), (11, 3)])
def test_block_noise_product_and_solves(n, n_remove):
    cfg, osys, pl, s, _ = _setup(n, n_remove)
    # P-a
    for v in (s, screens.random_vector(cfg, osys.Ns)):
        d_o = torch.empty(osys.Ns, dtype=torch.float32, device="cuda")
        pl.apply_css(dev(v), d_o)
        torch.cuda.synchronize()
        assert rel(d_o.cpu().numpy(), osys.apply_A(f32(v))) <= TOL_MVM
    # P-c
    n_it = 20
    _, h64 = osys.solve_cg(s, n_it)
    _, h32 = osys.solve_cg(s, n_it, dtype=np.float32)
    k_star = max(_horizon(h32, h64) - 2, 3)
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    assert pl.stats()["launches_last_solve"] > 4 * n_it                  # multi-kernel solver took over
    hg = pl.residuals(1, n_it)[0]
    assert np.abs(hg / h64 - 1.0)[:k_star + 1].max() <= TOL_TRAJ
    # P-d (CG and MINRES)
    zeta = osys.solve_direct(s)
    _, h = osys.solve_cg(s, 1000)
    n_conv = int(np.flatnonzero(h / h[0] < 1e-6)[0])
    pl.solve(dev(s), d_w, n_conv)
    torch.cuda.synchronize()
    assert rel(d_w.cpu().numpy(), osys.reconstruct(zeta, 0)) <= 1e-3
    pl.solve_minres(dev(s), d_w, 1, n_conv + 10)
    torch.cuda.synchronize()
    assert rel(d_w.cpu().numpy(), osys.reconstruct(zeta, 0)) <= 1e-3
    pl.close()


def test_block_noise_validation():
    cfg = small_lgs_config(n=8, n_gs=2, n_layers=2)
    nv = int(screens.subap_mask(cfg.n, cfg.obstruction).sum())
    diag = np.ones((2, 2, nv))
    bad = np.full((2, nv), 1.5)                                          # |sxy| > sqrt(sxx syy): not PSD
    with pytest.raises(tomo.TomoError) as e:
        tomo.TomoPlan(cfg, sigma2_subap=diag, sigma_xy_subap=bad, upload=False)
    assert e.value.code == tomo.TOMO_EINVAL
