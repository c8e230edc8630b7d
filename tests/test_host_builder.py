"""Row A0 on the CPU box: the library's host-side covariance-kernel builder (C++, include/tomo_host.h) against the
oracle's independent evaluation of the same paper formulas (Eq.50-53)."""
import math
import os
from dataclasses import replace

import numpy as np
import pytest

from oracle import toeplitz as tz
from oracle import vonkarman as vk
from paper_1806_07938_b200 import tomo
from tomo_inputs.configs import get_config, small_lgs_config, sweep_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _anchors():
    out = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "dphi_anchors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, val, r0, L0 = [t.strip() for t in line.split("|")]
        out[name] = (float(val), float(r0), float(L0))
    return out


def test_structure_function_matches_oracle_anchors_and_limits():
    a = _anchors()
    for name, (val, r0, L0) in a.items():
        if name.startswith("dphi_r"):
            got = tomo.host_structure_function(np.array([float(name[6:])]), r0, L0)[0]
            assert abs(got / val - 1) < 1e-10, name
    r = np.linspace(0.01, 120.0, 500)
    np.testing.assert_allclose(tomo.host_structure_function(r, 0.15, 25.0), vk.structure_function(r, 0.15, 25.0), rtol=1e-10)
    assert tomo.host_structure_function(np.array([0.0]), 0.15, 25.0)[0] == 0.0
    # saturation D(inf) = 0.17262866 (L0/r0)^{5/3} and the Kolmogorov limit 6.8839 (r/r0)^{5/3} for r << L0 (the C++ side
    # switches to the small-argument series there, reading G23)
    assert abs(tomo.host_structure_function(np.array([1e4]), 0.15, 25.0)[0] / a["dphi_inf"][0] - 1) < 1e-12
    got = tomo.host_structure_function(np.array([1e-3]), 0.15, 1e7)[0]
    assert abs(got / (6.8839 * (1e-3 / 0.15) ** (5.0 / 3.0)) - 1) < 1e-3


@pytest.mark.parametrize("n,nv,nvp", [(8, 52, 69), (16, 208, 241), (20, 316, 357), (32, 812, 877), (64, 3228, 3357),
                                       (74, 4304, 4453)])
def test_valid_counts(n, nv, nvp):
    """Centre-in-pupil / corner rule (Fig.2, reading G12): the counts of the configs ("~52", "~4300")."""
    sz = tomo.host_sizes(sweep_config(n))
    assert (sz["n_vs"], sz["n_vphi"]) == (nv, nvp)


def test_sizes_of_the_configs():
    assert tomo.host_sizes(get_config("cfg1"), 16, 16) == dict(n_vs=52, n_vphi=69, n_prime=9, P=16, P_os=16, Kp=1)
    s2 = tomo.host_sizes(get_config("cfg2"))
    assert (s2["n_prime"], s2["P"], s2["P_os"], s2["Kp"]) == (27, 40, 48, 7)
    s3 = tomo.host_sizes(get_config("cfg3"))          # automatic: next even 5-smooth size >= 2n-1 = 147
    assert (s3["n_prime"], s3["P"], s3["P_os"], s3["Kp"]) == (105, 150, 180, 35)
    c3 = get_config("cfg3")                            # BASELINE.json fixes the pad of cfg3 at 160
    assert tomo.host_sizes(c3, c3.pad, c3.pad_os)["P"] == 160
    assert [tomo.host_sizes(sweep_config(n))["P"] for n in (16, 32, 64, 96, 128)] == [32, 64, 128, 192, 256]
    assert [tomo.host_sizes(sweep_config(n))["P_os"] for n in (16, 32, 64, 96, 128)] == [40, 80, 160, 240, 320]
    assert [tomo.host_sizes(sweep_config(n))["n_prime"] for n in (16, 32, 64, 96, 128)] == [25, 47, 91, 135, 179]


def _oracle_generators(cfg, mname):
    dirs = [(w.ax, w.ay) for w in cfg.wfs]
    hgs = cfg.wfs[0].h_gs
    N, n = len(dirs), cfg.n
    th = tz.css_generators(n, cfg.d, dirs, hgs, cfg.h, cfg.frac, cfg.r0, cfg.L0, mname).reshape(2 * N, 2 * N, 2 * n - 1, 2 * n - 1)
    sz = tomo.host_sizes(cfg)
    xi = tz.cos_generators(n, sz["n_prime"], cfg.d, dirs, hgs, cfg.targets[0], cfg.h, cfg.frac, cfg.r0, cfg.L0, mname)
    if math.isinf(hgs):
        xi = xi.sum(axis=0, keepdims=True)        # NGS: layers share one grid and are summed (Eq.15)
    return th, xi.reshape(xi.shape[0], 2 * N, xi.shape[-1], xi.shape[-1])


@pytest.mark.parametrize("model", [tomo.TOMO_HUDGIN, tomo.TOMO_FRIED])
@pytest.mark.parametrize("name", ["cfg1", "small_lgs"])
def test_generators_match_oracle(name, model):
    cfg = get_config("cfg1") if name == "cfg1" else small_lgs_config(n=9, n_gs=3, n_layers=3, targets=((5.0, -3.0),))
    th, xi = _oracle_generators(cfg, {tomo.TOMO_HUDGIN: "hudgin", tomo.TOMO_FRIED: "fried"}[model])
    g = tomo.host_css_generators(cfg, model)
    assert np.abs(g - th).max() <= 1e-11 * np.abs(th).max()
    g2 = tomo.host_cos_generators(cfg, 0, model)
    assert g2.shape == xi.shape
    assert np.abs(g2 - xi).max() <= 1e-11 * np.abs(xi).max()


@pytest.mark.parametrize("model", [tomo.TOMO_HUDGIN, tomo.TOMO_FRIED])
@pytest.mark.parametrize("name", ["cfg1", "small_lgs"])
def test_layered_plan_generators_and_grid_edge_match_oracle(name, model):
    """Layered (MCAO) plans, L199 / reading G31: n_m from the field radius and the per-layer generators on the axis-centred
    n_m grid (NGS systems keep their layers apart too) against oracle/layered.py + toeplitz.cos_generators at beta = 0."""
    from oracle import layered as lay
    cfg = (replace(get_config("cfg1"), h=(0.0, 4000.0, 11000.0), frac=(0.55, 0.25, 0.2)) if name == "cfg1"
           else small_lgs_config(n=9, n_gs=3, n_layers=3))
    mname = {tomo.TOMO_HUDGIN: "hudgin", tomo.TOMO_FRIED: "fried"}[model]
    dirs, hgs = [(w.ax, w.ay) for w in cfg.wfs], cfg.wfs[0].h_gs
    for fov in (0.0, 25.0, 60.0):
        n_m, g = tomo.host_layer_generators(cfg, fov, model)
        assert n_m == lay.n_meta(cfg.n, cfg.d, cfg.h, hgs, fov)
        xi = tz.cos_generators(cfg.n, n_m, cfg.d, dirs, hgs, (0.0, 0.0), cfg.h, cfg.frac, cfg.r0, cfg.L0, mname)
        xi = xi.reshape(len(cfg.h), 2 * len(dirs), xi.shape[-1], xi.shape[-1])
        assert g.shape == xi.shape and np.abs(g - xi).max() <= 1e-11 * np.abs(xi).max()
    assert tomo.host_layer_generators(cfg, 0.0, model)[0] == tomo.host_sizes(cfg)["n_prime"]


@pytest.mark.parametrize("name", ["cfg1", "small_lgs"])
def test_fft_model_generators_discretisation_error_against_the_continuous_oracle(name, monkeypatch):
    """TOMO_FFTMODEL (Eq.41-46): the builder evaluates the Fourier integrals by 2-D FFTs on a grid of pixel w / 4, i.e. cut at
    |f| < 2 / w.  (i) Its FFT machinery reproduces the same Riemann sum written out directly (tests/fourier_sum.py) to 1e-9.
    (ii) Against the ORACLE -- the continuous integral, evaluated in physical space, sharing no grid with the builder -- the
    error is the truncated tail of sinc^2: ~0.2 % of the slope variance whatever w, r0 (both scale as r0^-5/3 w^-1/3; DESIGN.md
    G29); gated at 0.5 %."""
    import fourier_sum as fs
    from oracle import fftmodel as fm
    cfg = get_config("cfg1") if name == "cfg1" else small_lgs_config(n=9, n_gs=3, n_layers=3, targets=((5.0, -3.0),))
    g = tomo.host_css_generators(cfg, tomo.TOMO_FFTMODEL)
    g2 = tomo.host_cos_generators(cfg, 0, tomo.TOMO_FFTMODEL)
    th, xi = _oracle_generators(cfg, "fft")                                   # continuous integral
    var = th[0, 0, cfg.n - 1, cfg.n - 1]
    e_ss, e_ps = np.abs(g - th).max() / var, np.abs(g2 - xi).max() / np.abs(xi).max()
    print(f"[FFT model, {name}] builder vs continuous oracle: Sigma_ss {e_ss:.2e} of the variance, Sigma_phi-s {e_ps:.2e} of its maximum")
    assert e_ss <= 5e-3 and e_ps <= 5e-3
    monkeypatch.setattr(fm, "cov_slope_slope", lambda d, a, b, w, c, r0, L0: fs.cov_slope_slope(d, a, b, w, c, r0, L0, 512, 4))
    monkeypatch.setattr(fm, "cov_phase_slope", lambda d, b, w, c, r0, L0: fs.cov_phase_slope(d, b, w, c, r0, L0, 512, 4))
    th_g, xi_g = _oracle_generators(cfg, "fft")                               # the same sum on the builder's grid
    assert np.abs(g - th_g).max() <= 1e-9 * np.abs(th_g).max()
    assert np.abs(g2 - xi_g).max() <= 1e-9 * np.abs(xi_g).max()


def test_fft_model_generators_at_elt_geometry_against_the_continuous_oracle():
    """cfg3 geometry (n = 74, d = 0.5135 m, two opposite LGS of the 45" ring, layers up to 25 km): the builder's grid edge is
    1024 here (lags up to 73 plus the guide-star shift h_k d_alpha, which enters as a phase ramp, plus one outer scale to the
    nearest alias).  Sampled lags of the cross-WFS blocks against the continuous oracle: same 0.5 % gate, no wrap-around."""
    from dataclasses import replace
    from oracle import fftmodel as fm
    from oracle import geometry as geo
    from tomo_inputs.configs import WFS
    c3 = get_config("cfg3")
    cfg = replace(c3, wfs=(WFS(45.0, 0.0, 90e3, 2), WFS(-45.0, 0.0, 90e3, 2)), h=(0.0, 12500.0, 25000.0), frac=(0.5, 0.3, 0.2))
    g = tomo.host_css_generators(cfg, tomo.TOMO_FFTMODEL)
    n, d = cfg.n, cfg.d
    rng = np.random.default_rng(74)
    lags = np.concatenate([[[0, 0], [n - 1, n - 1], [-(n - 1), 0], [1, 0], [0, -1]], rng.integers(-(n - 1), n, size=(25, 2))])
    var = g[0, 0, n - 1, n - 1]
    worst = 0.0
    for (i, j) in ((0, 0), (0, 1)):
        for a in range(2):
            for b in range(2):
                want = np.zeros(len(lags))
                for hk, fk in zip(cfg.h, cfg.frac):
                    gam = geo.cone_factor(hk, 90e3)
                    sh = hk * (np.array([cfg.wfs[j].ax, cfg.wfs[j].ay]) - np.array([cfg.wfs[i].ax, cfg.wfs[i].ay])) * geo.ARCSEC
                    delta = gam * d * lags.astype(np.float64) + sh[None, :]
                    want += fk * fm.cov_slope_slope(delta, a, b, gam * d, 1.0 / d, cfg.r0, cfg.L0)
                got = g[2 * i + a, 2 * j + b, lags[:, 1] + n - 1, lags[:, 0] + n - 1]
                worst = max(worst, float(np.abs(got - want).max() / var))
    print(f"[FFT model, cfg3 geometry, grid edge 1024] builder vs continuous oracle: {worst:.2e} of the variance")
    assert worst <= 5e-3


@pytest.mark.parametrize("P", [16, 20, 30, 48])
def test_generator_spectrum_is_the_scaled_rfft2_of_the_embedding(P):
    rng = np.random.default_rng(5)
    n_in, n_out = 7, 9
    g = rng.standard_normal((n_in + n_out - 1, n_in + n_out - 1))
    sp = tomo.host_generator_spectrum(g, n_out, n_in, P)
    ref = np.fft.rfft2(tz.embed_generator(g, n_in, n_out, P)) / P ** 2      # [ky][kx]
    np.testing.assert_allclose(sp, ref.T, atol=1e-14 * np.abs(ref).max() * P)


def test_slab_segments_cover_every_pass_once_and_balance():
    """Host table of the persistent solver's batch path (include/tomo_host.h: tomo_host_slab_segments)."""
    for Ph, F, G in [(81, 1, 148), (81, 2, 148), (81, 3, 148), (81, 4, 148), (81, 16, 148), (81, 5, 148), (97, 16, 148),
                     (129, 16, 148), (129, 7, 148), (65, 16, 148), (9, 16, 148), (21, 16, 148), (11, 5, 148), (81, 16, 81)]:
        seg = tomo.host_slab_segments(Ph, F, G)
        seen = np.zeros((Ph, F), dtype=int)
        load = np.zeros(G, dtype=int)
        for b in range(G):
            f_lo, f_hi, kx2, g_lo, g_hi = (int(v) for v in seg[b, :5])
            assert 0 <= f_lo <= f_hi <= F and 0 <= g_lo <= g_hi <= F and 0 <= kx2 < Ph
            seen[b % Ph, f_lo:f_hi] += 1
            seen[kx2, g_lo:g_hi] += 1
            load[b] = (f_hi - f_lo) + (g_hi - g_lo)
            if g_hi > g_lo:
                assert kx2 != b % Ph                                  # a helped slab is somebody else's
        assert np.all(seen == 1), (Ph, F, G)                          # every (k_x, frame) pass exactly once
        target = -(-Ph * F // G)
        unbalanced = max(-(-F // ((G - 1 - kx) // Ph + 1)) for kx in range(Ph))
        assert load.max() <= unbalanced                               # never worse than without helpers
        if (Ph, F, G) in [(81, 16, 148), (81, 4, 148), (81, 3, 148), (97, 16, 148)]:
            assert load.max() == target < unbalanced, (Ph, F, G, load.max(), target)
        if F == 1:
            assert load.max() == 1 and not np.any(seg[:, 4] > seg[:, 3])
