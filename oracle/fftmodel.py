"""FFT slope model (App. A.A of the paper, Eq.41-46) (oracle, fp64).  Test infrastructure only.

The SH-WFS slope is the phase gradient AVERAGED over the subaperture (Eq.41).  Eq.43 (L545) and Eq.46 (L566) write
its covariances as Fourier integrals of the von Karman spectrum Phi_phi (Eq.45) filtered by the subaperture
H(f) = sinc(w f_x) sinc(w f_y) (Eq.44); "in actual computation, the FFT covariance model is computed by the FFT, and
its actual accuracy depends on the sampling" (L572).  What the model DEFINES is the continuous integral; this oracle
evaluates that integral by a route that shares nothing with an FFT or its frequency grid: in physical space.

By the fundamental theorem of calculus the x-gradient averaged over a square subaperture of edge w centred on r is the
difference of the phase averaged over its two edges x = r_x +- w/2,
    s_x(r) = c [ <phi>_(+) - <phi>_(-) ],   <phi>_(+-) = 1/w int_{-w/2}^{w/2} phi(r_x +- w/2, r_y + y) dy,
c = 1/d (this repository's slope unit rad/m, reading G6; with the cone compression w = gamma d of an LGS layer a pupil-plane
gradient is gamma times the layer-plane one: c w = gamma, reading G29).  With E[(a-b)(c'-d')] = 1/2 [D(a,d') + D(b,c') -
D(a,c') - D(b,d')] for phase differences and D = D_phi of Eq.53 (vonkarman.py, pinned on its own) this gives, for a
separation Delta = (second position) - (first position) as everywhere in oracle/:

    cov(s_x, s_x)(Delta) = c^2 int_{-w}^{w} (w - |u|)/w^2 [ 1/2 D(Dx + w, Dy + u) + 1/2 D(Dx - w, Dy + u) - D(Dx, Dy + u) ] du
    cov(s_x, s_y)(Delta) = c^2/(2 w^2) int int_{[-w/2, w/2]^2} [ D(Dx + x' - w/2, Dy - w/2 - y) + D(Dx + x' + w/2, Dy + w/2 - y)
                                                                - D(Dx + x' - w/2, Dy + w/2 - y) - D(Dx + x' + w/2, Dy - w/2 - y) ] dx' dy
    cov(phi, s_x)(Delta) = -c/(2 w) int_{-w/2}^{w/2} [ D(Dx + w/2, Dy + y) - D(Dx - w/2, Dy + y) ] dy
(y-slopes: x and y exchanged), i.e. the two-point Hudgin-like forms of Eq.50-52 with every phase sample replaced by an edge
average -- which is exactly what multiplying the spectrum by H^2 (Eq.43) or H (Eq.46) does.  The integrals are taken by
Gauss-Legendre panels split where D's r^(5/3) cusp can fall inside the range (converged to ~1e-8 of the slope variance, test_oracle_fftmodel).

The library's builder evaluates the same model by a 2-D FFT over a truncated frequency grid (G29); its
discretisation error against this oracle is measured in tests/test_host_builder.py, not assumed.
"""
import numpy as np

from . import vonkarman as vk

N_NODES_1D = 24          # Gauss-Legendre nodes per panel of the 1-D integrals (converged to 1e-8: test_oracle_fftmodel)
N_NODES_2D = 12          # ... per panel and axis of the 2-D integral

_GL = {}


def _gl(n):
    if n not in _GL:
        _GL[n] = np.polynomial.legendre.leggauss(n)
    return _GL[n]


def _panels(lo, hi, breaks, n):
    """Nodes and weights of Gauss-Legendre panels on [lo, hi] split at the (clipped) break points, per row of `breaks`
    ([M][nb]): returns x [M][(nb + 1) n], w [M][(nb + 1) n].  Zero-length panels carry zero weight."""
    t, wt = _gl(n)
    b = np.clip(np.asarray(breaks, dtype=np.float64), lo, hi)
    edges = np.sort(np.concatenate([np.full((b.shape[0], 1), lo), b, np.full((b.shape[0], 1), hi)], axis=1), axis=1)
    a, c = edges[:, :-1], edges[:, 1:]                        # [M][nb + 1]
    mid, half = 0.5 * (a + c), 0.5 * (c - a)
    x = mid[:, :, None] + half[:, :, None] * t[None, None, :]
    w = half[:, :, None] * wt[None, None, :]
    return x.reshape(x.shape[0], -1), w.reshape(w.shape[0], -1)


def _D(dx, dy, r0, L0):
    return vk.structure_function(np.hypot(dx, dy), r0, L0)


def _unique(delta):
    flat = np.ascontiguousarray(np.asarray(delta, dtype=np.float64).reshape(-1, 2))
    uniq, inv = np.unique(np.round(flat, 12), axis=0, return_inverse=True)
    return uniq, inv.reshape(-1)


def _same_axis(dpar, dperp, w, c, r0, L0):
    """cov of two slopes along the SAME axis: dpar = separation along that axis, dperp across it."""
    u, wu = _panels(-w, w, np.stack([np.zeros_like(dperp), -dperp], axis=1), N_NODES_1D)
    tri = (w - np.abs(u)) / (w * w)
    a = dpar[:, None]
    g = 0.5 * _D(a + w, dperp[:, None] + u, r0, L0) + 0.5 * _D(a - w, dperp[:, None] + u, r0, L0) - _D(a, dperp[:, None] + u, r0, L0)
    return c * c * np.sum(wu * tri * g, axis=1)


def _cross_axis(dx, dy, w, c, r0, L0, chunk=256):
    """cov(s_x at the first position, s_y at the second), separation (dx, dy) = second - first."""
    out = np.empty(dx.shape[0])
    h = 0.5 * w
    for i0 in range(0, dx.shape[0], chunk):
        ax, ay = dx[i0:i0 + chunk], dy[i0:i0 + chunk]
        xs, wx = _panels(-h, h, np.stack([-ax - h, -ax + h], axis=1), N_NODES_2D)        # x' : where Dx + x' -+ w/2 = 0
        ys, wy = _panels(-h, h, np.stack([ay - h, ay + h], axis=1), N_NODES_2D)          # y  : where Dy -+ w/2 - y = 0
        X = ax[:, None, None] + xs[:, :, None]
        Y = ay[:, None, None] - ys[:, None, :]
        g = _D(X - h, Y - h, r0, L0) + _D(X + h, Y + h, r0, L0) - _D(X - h, Y + h, r0, L0) - _D(X + h, Y - h, r0, L0)
        out[i0:i0 + chunk] = np.einsum("mi,mj,mij->m", wx, wy, g)
    return (c * c / (2.0 * w * w)) * out


def cov_slope_slope(delta, a: int, b: int, width: float, c: float, r0: float, L0: float):
    """cov(s_a(r), s_b(r + Delta)) of the subaperture-averaged gradient (Eq.43), Delta [..., 2] in metres."""
    delta = np.asarray(delta, dtype=np.float64)
    uq, inv = _unique(delta)
    dx, dy = uq[:, 0], uq[:, 1]
    if a == 0 and b == 0:
        val = _same_axis(dx, dy, width, c, r0, L0)
    elif a == 1 and b == 1:
        val = _same_axis(dy, dx, width, c, r0, L0)
    elif a == 0:
        val = _cross_axis(dx, dy, width, c, r0, L0)
    else:                                   # cov(s_y(r), s_x(r + D)) = cov(s_x(r'), s_y(r' - D))
        val = _cross_axis(-dx, -dy, width, c, r0, L0)
    return val[inv].reshape(delta.shape[:-1])


def cov_phase_slope(delta, b: int, width: float, c: float, r0: float, L0: float):
    """cov(phi(r_p), s_b(r_p + Delta)) (Eq.46): the phase sample against the two edge averages."""
    delta = np.asarray(delta, dtype=np.float64)
    uq, inv = _unique(delta)
    dpar, dperp = (uq[:, 0], uq[:, 1]) if b == 0 else (uq[:, 1], uq[:, 0])
    h = 0.5 * width
    y, wy = _panels(-h, h, (-dperp)[:, None], N_NODES_1D)
    g = _D(dpar[:, None] + h, dperp[:, None] + y, r0, L0) - _D(dpar[:, None] - h, dperp[:, None] + y, r0, L0)
    val = (-c / (2.0 * width)) * np.sum(wy * g, axis=1)
    return val[inv].reshape(delta.shape[:-1])
