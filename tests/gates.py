"""Shared comparison gates of the GPU parity tests.

Every vector comparison is gated twice: the relative L2 norm of the difference AND the largest element-wise difference
in units of the rms of the expected vector (a relative L2 norm alone lets a 1 % error on ONE edge subaperture of a
51 648-vector through a 1e-4 gate: it contributes 4e-5).
"""
import numpy as np

TOL_MAX_PRODUCT = 1e-5      # products and teacher-forced steps (fp32, measured ~1e-6): max |diff| <= 1e-5 rms


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def max_abs(a, b):
    """max |a - b| in units of the rms of b."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    rms = float(np.sqrt(np.mean(b ** 2)))
    return float(np.max(np.abs(a - b)) / rms) if rms > 0 else float(np.max(np.abs(a - b)))


def assert_close(got, want, tol_l2, tol_max=None, what=""):
    """rel-L2 <= tol_l2 and max-abs <= tol_max (default: 1e-5 rms for the 1e-4 product / step gates, 10 x tol_l2 for the
    trajectory gates, whose legitimate deviation is not uniform over the elements).  Returns (rel-L2, max-abs)."""
    if tol_max is None:
        tol_max = TOL_MAX_PRODUCT if tol_l2 <= 1e-4 else 10.0 * tol_l2
    e2, em = rel(got, want), max_abs(got, want)
    assert e2 <= tol_l2 and em <= tol_max, (what, "rel-L2", e2, "max-abs/rms", em, "gates", tol_l2, tol_max)
    return e2, em
