"""Mode-removal projectors (oracle, fp64).  Test infrastructure only.

Eq.36: M_{s,i} = I - Z_{s,i} Z_{s,i}^+, Z_{s,i} the tip/tilt/focus modal
matrix over the valid subapertures of WFS i (L323); M_s = blockdiag(M_{s,i}) (L327).
Readings (G14): slope-space columns are tip = (1 on x-slopes, 0 on y-slopes),
tilt = (0, 1), focus = (x_q, y_q) (the gradient of x^2+y^2 up to a factor); Z^+ is the
Moore-Penrose pseudo-inverse so M is the orthogonal projector onto range(Z)^perp.
Phase space: Z_phi = [1, x_p, y_p (, x_p^2 + y_p^2)] over the valid phase points (piston is
added to the paper's three columns); NGS-only systems remove piston only.
"""
import numpy as np


def slope_modes(centres_valid, n_remove: int):
    """Z_{s,i}: (2 n_vs, n_remove), rows ordered [x-slopes; y-slopes]."""
    nv = centres_valid.shape[0]
    cols = []
    if n_remove >= 2:
        cols.append(np.concatenate([np.ones(nv), np.zeros(nv)]))
        cols.append(np.concatenate([np.zeros(nv), np.ones(nv)]))
    if n_remove >= 3:
        cols.append(np.concatenate([centres_valid[:, 0], centres_valid[:, 1]]))
    if not cols:
        return np.zeros((2 * nv, 0))
    return np.stack(cols, axis=1)


def removal_matrix(Z):
    """I - Z Z^+  (Eq.36)."""
    m = Z.shape[0]
    if Z.shape[1] == 0:
        return np.eye(m)
    return np.eye(m) - Z @ np.linalg.pinv(Z)


def slope_projector(centres_valid, n_remove_per_wfs):
    """M_s = blockdiag_i(M_{s,i})  (L327)."""
    nv = centres_valid.shape[0]
    N = len(n_remove_per_wfs)
    M = np.zeros((N * 2 * nv, N * 2 * nv))
    for i, nr in enumerate(n_remove_per_wfs):
        Mi = removal_matrix(slope_modes(centres_valid, nr))
        M[i * 2 * nv:(i + 1) * 2 * nv, i * 2 * nv:(i + 1) * 2 * nv] = Mi
    return M


def phase_modes(phase_pts_valid, n_remove: int):
    """Z_phi: piston (always) + tip/tilt (n_remove>=2) + focus (n_remove>=3)."""
    x, y = phase_pts_valid[:, 0], phase_pts_valid[:, 1]
    cols = [np.ones_like(x)]
    if n_remove >= 2:
        cols += [x, y]
    if n_remove >= 3:
        cols += [x * x + y * y]
    return np.stack(cols, axis=1)


def phase_projector(phase_pts_valid, n_remove: int):
    return removal_matrix(phase_modes(phase_pts_valid, n_remove))
