"""Low-order NGS path on the GPU (NEXT rank 5; reading G30): tomo_lo_apply against the oracle's add-back, element by element."""
from dataclasses import replace

import numpy as np
import pytest

from oracle import geometry as geo
from oracle import loworder as olo
from tomo_inputs.configs import BASE_SEED, WFS, get_config

pytestmark = pytest.mark.gpu

LO3 = (WFS(40.0, 10.0), WFS(-25.0, 35.0), WFS(-10.0, -45.0))


def _case(name, targets, n_frames, seed):
    import torch
    from paper_1806_07938_b200 import tomo
    cfg = replace(get_config(name), lo_wfs=LO3, targets=targets)
    if name == "cfg2":          # the oracle is O(n_vs^2) per covariance entry: two sensors, one layer at this size
        cfg = replace(cfg, lo_wfs=LO3[:2], h=(6000.0,), frac=(1.0,))
    d = cfg.D / cfg.n
    sm = geo.subap_mask(cfg.n, cfg.D, cfg.obstruction)
    cv = geo.subap_centres(cfg.n, d)[sm.ravel()]
    pts = geo.phase_points(cfg.n, d)[geo.phase_mask(sm).ravel()]
    sigma2 = 0.2
    Ro = olo.lo_estimator(cv, d, [(w.ax, w.ay) for w in cfg.lo_wfs], targets, cfg.h, cfg.frac, cfg.r0, cfg.L0, sigma2)
    rng = np.random.default_rng(BASE_SEED + seed)
    g = rng.standard_normal((n_frames, len(cfg.lo_wfs), 2)) * 3.0             # mean slopes [rad/m]
    w0 = rng.standard_normal((n_frames, len(targets), pts.shape[0]))   # stands for the high-order wavefront
    want = w0 + np.stack([olo.lo_addback(Ro, g[f], pts) for f in range(n_frames)])
    lo = tomo.LowOrder(cfg, sigma2)
    wd = torch.tensor(w0, dtype=torch.float32, device="cuda")
    gd = torch.tensor(g, dtype=torch.float32, device="cuda")
    lo.apply(gd, wd)
    torch.cuda.synchronize()
    got = wd.cpu().numpy().astype(np.float64)
    lo.close()
    return got, want, w0


@pytest.mark.parametrize("name,targets,n_frames", [
    ("cfg1", ((0.0, 0.0),), 1),
    ("cfg2", ((0.0, 0.0), (20.0, -5.0)), 5),                      # 357 phase points: two blocks, ragged tail
])
def test_lo_apply_equals_oracle(name, targets, n_frames):
    got, want, w0 = _case(name, targets, n_frames, 77)
    # fp32 path: R_lo, coordinates and the data are rounded to fp32, two FMAs per point
    assert np.abs(got - want).max() <= 2e-6 * np.abs(want).max()
    assert np.abs(got - w0).max() > 1e-2 * np.abs(want).max()       # the tilt was really added


def test_lo_apply_zero_frames_and_bad_arguments():
    import torch
    from paper_1806_07938_b200 import tomo
    cfg = replace(get_config("cfg1"), lo_wfs=LO3)
    lo = tomo.LowOrder(cfg, 0.1)
    w = torch.ones((0, 1, 69), dtype=torch.float32, device="cuda")
    g = torch.ones((0, 3, 2), dtype=torch.float32, device="cuda")
    lo.apply(g, w)                                                  # n_frames == 0: no launch, no error
    with pytest.raises(ValueError):
        lo.apply(torch.ones((2, 2, 2), dtype=torch.float32, device="cuda"), torch.ones((2, 1, 69), dtype=torch.float32, device="cuda"))
    lo.close()


def test_lo_apply_full_size_cfg4_batch16():
    """cfg4 geometry (4453 valid phase points, 10 targets, 3 sensors), 16 frames: every output against the oracle's add-back.
    The pair-by-pair oracle cannot build R_lo at this size, so R_lo here is the library's host builder's (gated against the
    oracle at small sizes and by its full-size properties in tests/test_host_loworder.py); the kernel under test only applies it."""
    import torch
    from paper_1806_07938_b200 import tomo
    cfg = get_config("cfg4")
    d = cfg.D / cfg.n
    sm = geo.subap_mask(cfg.n, cfg.D, cfg.obstruction)
    pts = geo.phase_points(cfg.n, d)[geo.phase_mask(sm).ravel()]
    R, _ = tomo.host_lo_estimator(cfg, 0.05)
    rng = np.random.default_rng(BASE_SEED + 404)
    n_frames, T, n_lo = 16, len(cfg.targets), len(cfg.lo_wfs)
    g = rng.standard_normal((n_frames, n_lo, 2))
    w0 = rng.standard_normal((n_frames, T, pts.shape[0]))
    want = w0 + np.stack([olo.lo_addback(R, g[f], pts) for f in range(n_frames)])
    lo = tomo.LowOrder(cfg, 0.05)
    wd = torch.tensor(w0, dtype=torch.float32, device="cuda")
    lo.apply(torch.tensor(g, dtype=torch.float32, device="cuda"), wd)
    torch.cuda.synchronize()
    got = wd.cpu().numpy().astype(np.float64)
    lo.close()
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 2e-6 * np.abs(want).max()
