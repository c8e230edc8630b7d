"""Pins of oracle/loworder.py (reading G30: MMSE tip/tilt from aperture-mean NGS slopes; the paper is silent, L321/L412).

Each pin is something the mathematics fixes without the oracle's own formula:
  * telescoping: the Hudgin x-slopes of one row of contiguous subapertures sum to [phi(right edge) - phi(left edge)]/d
    (Eq.47), so on a full square grid var(mean s_x) is a double sum of D_phi over ROW pairs only (Eq.53);
  * a noiseless sensor in the target direction is returned unchanged (R_lo = I_2);
  * mirror symmetry of two sensors about the target; decorrelation far beyond L0; R_lo -> C_tau,g / sigma2 for large noise.
"""
import numpy as np

from oracle import geometry as geo
from oracle import loworder as lo
from oracle import vonkarman as vk

R0, L0 = 0.15, 25.0


def _valid(n, D):
    m = geo.subap_mask(n, D)
    return geo.subap_centres(n, D / n)[m.ravel()]


def test_mean_slope_variance_telescopes_to_edge_phase_differences():
    n, d = 6, 0.5
    centres = geo.subap_centres(n, d)                      # full square grid, every subaperture valid
    C = lo.mean_slope_covariance(centres, d, [(3.0, -2.0)], (0.0, 4000.0), (0.6, 0.4), R0, L0)
    rows = np.arange(n) * d
    dy = np.abs(rows[:, None] - rows[None, :])
    want = (vk.structure_function(np.hypot(n * d, dy), R0, L0) - vk.structure_function(dy, R0, L0)).sum() / (n * n * d) ** 2
    assert np.isclose(C[0, 0], want, rtol=1e-12)
    assert np.isclose(C[1, 1], want, rtol=1e-12)           # x <-> y symmetry of the square grid
    assert abs(C[0, 1]) < 1e-14 * want and abs(C[1, 0]) < 1e-14 * want


def test_two_directions_telescoping_with_layer_shift():
    n, d, hk, sep = 5, 0.4, 6000.0, 20.0                    # one layer, two sensors sep arcsec apart along y
    centres = geo.subap_centres(n, d)
    C = lo.mean_slope_covariance(centres, d, [(0.0, 0.0), (0.0, sep)], (hk,), (1.0,), R0, L0)
    rows = np.arange(n) * d
    dy = rows[None, :] + hk * sep * geo.ARCSEC - rows[:, None]
    want = (vk.structure_function(np.hypot(n * d, dy), R0, L0) - vk.structure_function(np.abs(dy), R0, L0)).sum() / (n * n * d) ** 2
    assert np.isclose(C[0, 2], want, rtol=1e-12) and np.isclose(C[2, 0], want, rtol=1e-12)
    assert np.allclose(C, C.T, rtol=0, atol=1e-12)
    assert np.linalg.eigvalsh(C).min() > 0


def test_noiseless_sensor_on_the_target_is_returned_unchanged():
    cv = _valid(8, 4.0)
    R = lo.lo_estimator(cv, 0.5, [(7.0, -3.0)], [(7.0, -3.0)], (0.0, 5000.0), (0.7, 0.3), R0, L0, 0.0)
    assert np.allclose(R, np.eye(2), atol=1e-10)


def test_mirror_symmetry_far_field_and_large_noise():
    cv = _valid(8, 4.0)
    h, f = (0.0, 5000.0, 10000.0), (0.5, 0.3, 0.2)
    R = lo.lo_estimator(cv, 0.5, [(15.0, 0.0), (-15.0, 0.0)], [(0.0, 0.0)], h, f, R0, L0, 1e-3)
    assert np.allclose(R[:, 0:2], R[:, 2:4], rtol=1e-10, atol=1e-14)      # equal weights for mirrored sensors
    assert abs(R[0, 1]) < 1e-12 and abs(R[1, 0]) < 1e-12                  # no x-y mixing on the mirror axis
    # one high layer, sensor 2 degrees away: shift 350 m >> L0 -> nothing to estimate from
    Rfar = lo.lo_estimator(cv, 0.5, [(7200.0, 0.0)], [(0.0, 0.0)], (10000.0,), (1.0,), R0, L0, 1e-6)
    Rnear = lo.lo_estimator(cv, 0.5, [(1.0, 0.0)], [(0.0, 0.0)], (10000.0,), (1.0,), R0, L0, 1e-6)
    assert np.abs(Rfar).max() < 1e-3 * np.abs(Rnear).max()
    big = 1e9
    Cm = lo.mean_slope_covariance(cv, 0.5, [(15.0, 0.0), (0.0, 0.0)], h, f, R0, L0)
    Rbig = lo.lo_estimator(cv, 0.5, [(15.0, 0.0)], [(0.0, 0.0)], h, f, R0, L0, big)
    assert np.allclose(Rbig * big, Cm[2:, :2], rtol=1e-6, atol=1e-10)


def test_addback_is_the_plane_through_the_estimated_tilt():
    n, d = 8, 0.5
    pts = geo.phase_points(n, d)[geo.phase_mask(geo.subap_mask(n, 4.0)).ravel()]
    R = np.array([[0.5, 0.1, 0.2, 0.0], [0.0, 0.4, -0.1, 0.3]])
    g = np.array([[1.0, 2.0], [-3.0, 0.5]])
    w = lo.lo_addback(R, g, pts)
    tx, ty = 0.5 * 1 + 0.1 * 2 + 0.2 * -3, 0.4 * 2 + 0.1 * 3 + 0.3 * 0.5
    assert w.shape == (1, pts.shape[0])
    # finite differences of the plane give back the tilt; zero mean over a symmetric pupil
    i0 = np.flatnonzero((pts[:, 0] == 0.0) & (pts[:, 1] == 0.0))[0]
    ix = np.flatnonzero((pts[:, 0] == d) & (pts[:, 1] == 0.0))[0]
    iy = np.flatnonzero((pts[:, 0] == 0.0) & (pts[:, 1] == d))[0]
    assert np.isclose((w[0, ix] - w[0, i0]) / d, tx) and np.isclose((w[0, iy] - w[0, i0]) / d, ty)
    assert abs(w.mean()) < 1e-12
