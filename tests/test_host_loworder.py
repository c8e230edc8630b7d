"""Low-order NGS path (NEXT rank 5; reading G30): the library's host builder against the oracle, no device needed.

The library sums cov_ab over LAGS weighted by the mask autocorrelation; the oracle averages the position-based covariance
over all PAIRS of valid subapertures.  Both in fp64: they must agree to rounding."""
from dataclasses import replace

import numpy as np
import pytest

from oracle import geometry as geo
from oracle import loworder as olo
from paper_1806_07938_b200 import tomo
from tomo_inputs.configs import WFS, get_config

LO3 = (WFS(40.0, 10.0), WFS(-25.0, 35.0), WFS(-10.0, -45.0))


def _oracle(cfg, sigma2, model="hudgin"):
    d = cfg.D / cfg.n
    cv = geo.subap_centres(cfg.n, d)[geo.subap_mask(cfg.n, cfg.D, cfg.obstruction).ravel()]
    lo_dirs = [(w.ax, w.ay) for w in cfg.lo_wfs]
    R = olo.lo_estimator(cv, d, lo_dirs, cfg.targets, cfg.h, cfg.frac, cfg.r0, cfg.L0, sigma2, model)
    Cm = olo.mean_slope_covariance(cv, d, lo_dirs + list(cfg.targets), cfg.h, cfg.frac, cfg.r0, cfg.L0, model)
    return R, Cm


@pytest.mark.parametrize("name,model", [("cfg1", "hudgin"), ("cfg1", "fried"), ("n14", "hudgin")])
def test_host_estimator_equals_oracle(name, model):
    cfg = replace(get_config("cfg1"), lo_wfs=LO3, targets=((0.0, 0.0), (20.0, -5.0), (-30.0, 30.0)))
    if name == "n14":           # larger grid with a central obstruction, three layers (the oracle is O(n_vs^2) per entry)
        cfg = replace(cfg, n=14, D=7.0, obstruction=0.3, pad=0, pad_os=0, h=(0.0, 4000.0, 11000.0), frac=(0.5, 0.3, 0.2))
    sigma2 = 0.3
    R, Cm = tomo.host_lo_estimator(cfg, sigma2, tomo.TOMO_FRIED if model == "fried" else tomo.TOMO_HUDGIN)
    Ro, Cmo = _oracle(cfg, sigma2, model)
    assert R.shape == (6, 6)
    scale = np.abs(Cmo).max()
    assert np.abs(Cm - Cmo).max() <= 1e-10 * scale
    assert np.abs(R - Ro).max() <= 1e-8 * np.abs(Ro).max()


def test_host_estimator_lgs_high_order_set_does_not_change_it():
    # the low-order sensors and the targets are at infinity: no cone factor, whatever the high-order guide stars are
    cfg = replace(get_config("cfg2"), lo_wfs=LO3[:1], h=(0.0, 8000.0), frac=(0.6, 0.4))
    R, _ = tomo.host_lo_estimator(cfg, 0.1)
    Ro, _ = _oracle(cfg, 0.1)
    assert np.abs(R - Ro).max() <= 1e-8 * np.abs(Ro).max()


def test_host_estimator_argument_errors():
    cfg = get_config("cfg1")
    with pytest.raises(tomo.TomoError) as e:
        tomo.host_lo_estimator(cfg, 0.1)                      # no low-order sensor
    assert e.value.code == tomo.TOMO_EINVAL
    cfg = replace(cfg, lo_wfs=LO3)
    with pytest.raises(tomo.TomoError) as e:
        tomo.host_lo_estimator(cfg, 0.1, tomo.TOMO_FFTMODEL)
    assert e.value.code == tomo.TOMO_EUNSUPPORTED
    with pytest.raises(tomo.TomoError) as e:
        tomo.host_lo_estimator(cfg, -1.0)
    assert e.value.code == tomo.TOMO_EINVAL
    with pytest.raises(tomo.TomoError) as e:                  # two coincident noiseless sensors: singular C_gg
        tomo.host_lo_estimator(replace(cfg, lo_wfs=(LO3[0], LO3[0])), 0.0)
    assert e.value.code == tomo.TOMO_EINVAL


def test_host_estimator_cfg4_full_size_properties():
    """cfg4 (74 x 74, 3 NGS tip/tilt sensors, 10 targets, 35 layers): too large for the pair-by-pair oracle, so properties that
    hold at any size: the covariance of the mean slopes is symmetric positive definite with equal diagonal blocks (every
    direction sees the same statistics), R_lo C_gg-weighted gains stay below one, and with no noise a target placed on a
    sensor takes that sensor's measurement."""
    cfg = get_config("cfg4")
    R, Cm = tomo.host_lo_estimator(cfg, 0.05)
    assert R.shape == (2 * len(cfg.targets), 2 * len(cfg.lo_wfs))
    assert np.abs(Cm - Cm.T).max() <= 1e-12 * np.abs(Cm).max()
    assert np.linalg.eigvalsh(Cm).min() > 0
    d0 = Cm[0:2, 0:2]
    for k in range(Cm.shape[0] // 2):
        assert np.allclose(Cm[2 * k:2 * k + 2, 2 * k:2 * k + 2], d0, rtol=1e-12, atol=1e-14 * np.abs(d0).max())
    gains = R[0::2, 0::2].sum(axis=1)              # x-tilt of each target from the x-slopes of all sensors
    assert np.all(gains > 0.0) and np.all(gains < 1.0)
    s0 = cfg.lo_wfs[0]
    R0, _ = tomo.host_lo_estimator(replace(cfg, lo_wfs=(s0,), targets=((s0.ax, s0.ay),)), 0.0)
    assert np.allclose(R0, np.eye(2), atol=1e-10)
