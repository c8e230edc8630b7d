"""Offline reconstructor columns through the batch path (NEXT rank 4): R = M_phi W_phi Sigma_phi-s A^+ M_s built
one unit right-hand side per frame, against the dense oracle's explicit matrix, and R s against the direct path."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1806_07938_b200 import tomo  # noqa: E402
from paper_1806_07938_b200.reconstructor import reconstructor_columns  # noqa: E402
from test_gpu_parity import dev, f32, make_plan, rel, system  # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,solver", [("cfg1", tomo.TOMO_SOLVER_PERSISTENT), ("small_lgs", tomo.TOMO_SOLVER_PERSISTENT),
                                         ("small_lgs", tomo.TOMO_SOLVER_MULTIKERNEL)])
def test_reconstructor_columns_match_the_dense_oracle(name, solver):
    cfg, _, osys, data = system(name)
    # dense R of the oracle: M_phi C_os M_s A^+ M_s  (A^+ through the symmetric eigen-decomposition)
    w, V = np.linalg.eigh((osys.A + osys.A.T) * 0.5)
    keep = w > w.max() * 1e-10
    Apinv = (V[:, keep] / w[keep]) @ V[:, keep].T
    R_or = np.vstack([osys.Mphi @ (osys.Cos[t] @ (osys.Ms @ Apinv @ osys.Ms)) for t in range(len(cfg.targets))])
    pl = make_plan(name, max_batch=16, solver=solver)
    rng = np.random.default_rng(5)
    cols = sorted(rng.choice(osys.Ns, size=40, replace=False).tolist())
    # iterations until the ORACLE's CG has converged (1e-6) on unit right-hand sides (a fixed-count fp32 CG run far beyond
    # convergence drifts again: the count is part of the workload, as in gate P-d)
    n_it = 0
    for j in cols[:6]:
        e = np.zeros(osys.Ns); e[j] = 1.0
        _, h = osys.solve_cg(e, 600)
        n_it = max(n_it, int(np.flatnonzero(h / h[0] < 1e-6)[0]))
    R = reconstructor_columns(pl, n_it, cols).cpu().numpy().astype(np.float64)       # [col][T * n_vphi]
    want = R_or[:, cols].T
    assert rel(R, want) <= 1e-3, rel(R, want)
    worst = max(rel(R[i], want[i]) for i in range(len(cols)))
    assert worst <= 5e-3, worst
    # MINRES columns agree as well
    Rm = reconstructor_columns(pl, n_it, cols[:16], minres=True).cpu().numpy().astype(np.float64)
    assert rel(Rm, want[:16]) <= 1e-3
    pl.close()


def test_full_reconstructor_times_slopes_equals_the_direct_path():
    cfg, _, osys, data = system("cfg1")
    pl = make_plan("cfg1", max_batch=16)
    n_it = 150
    R = reconstructor_columns(pl, n_it)                                             # all 208 columns, 13 batched solves
    s = f32(data["slopes"][0].ravel())
    d_w = torch.empty(pl.wavefront_len, dtype=torch.float32, device="cuda")
    pl.solve(dev(s), d_w, n_it)
    torch.cuda.synchronize()
    via_R = (R.double().T @ dev(s, torch.float64)).cpu().numpy()
    assert rel(via_R, d_w.cpu().numpy().astype(np.float64)) <= 1e-3
    assert rel(via_R, osys.reconstruct(osys.solve_direct(s), 0)) <= 1e-3
    pl.close()
