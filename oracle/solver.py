"""Direct and iterative solution of Eq.12 (oracle).  Test infrastructure only.

Direct: zeta* = A^+ b with A = M_s (W_s Sigma_ss W_s^T + Sigma_eta) M_s^T (Eq.34);
A is singular on range(Z) when modes are removed, hence the symmetric pseudo-inverse
(Cholesky when nothing is removed).

CG: the textbook Hestenes-Stiefel recurrence the paper names in S2.G (L337, refs [19,20]),
cold start (L490 "zero initial vector"), no preconditioner, a fixed number of iterations
(reading G16):
    x0 = 0 (or a warm start), r0 = b - A x0, p0 = r0, rho0 = r0.r0
    q = A p; alpha = rho/(p.q); x += alpha p; r -= alpha q; rho' = r.r; beta = rho'/rho;
    p = r + beta p; rho = rho'
The history is sqrt(rho_k), k = 0..n_iter (the recurrence residual).
"""
import numpy as np
import scipy.linalg as sla


def direct_solve(A, b, singular: bool):
    if not singular:
        cf = sla.cho_factor(A)
        return sla.cho_solve(cf, b)
    # symmetric pseudo-inverse through the eigen-decomposition; null space = range(Z)
    w, V = np.linalg.eigh((A + A.T) * 0.5)
    tol = w.max() * A.shape[0] * np.finfo(np.float64).eps * 16
    inv = np.where(w > tol, 1.0 / np.where(w > tol, w, 1.0), 0.0)
    return V @ (inv * (V.T @ b))


def cg(apply_A, b, n_iter: int, x0=None, dtype=np.float64, record=False):
    """Fixed-count CG.  apply_A: callable v -> A v (any precision handling is the caller's).
    Returns x, history[n_iter+1], and (if record) the per-iteration states and scalars."""
    b = np.asarray(b, dtype=dtype)
    if x0 is None:
        x = np.zeros_like(b)
        r = b.copy()
    else:
        x = np.asarray(x0, dtype=dtype).copy()
        r = (b - apply_A(x)).astype(dtype)
    p = r.copy()
    rho = dtype(r @ r)
    hist = [float(np.sqrt(rho))]
    states = []
    for _ in range(n_iter):
        if record:
            states.append(dict(x=x.copy(), r=r.copy(), p=p.copy(), rho=float(rho)))
        q = np.asarray(apply_A(p), dtype=dtype)
        pq = dtype(p @ q)
        if rho == 0 or pq <= 0:      # breakdown: freeze (reading G16)
            alpha = dtype(0)
            beta = dtype(0)
            rho_new = rho
        else:
            alpha = dtype(rho / pq)
            x = (x + alpha * p).astype(dtype)
            r = (r - alpha * q).astype(dtype)
            rho_new = dtype(r @ r)
            beta = dtype(rho_new / rho)
            p = (r + beta * p).astype(dtype)
        if record:
            states[-1].update(alpha=float(alpha), beta=float(beta), q=q.copy())
        rho = rho_new
        hist.append(float(np.sqrt(rho)))
    hist = np.asarray(hist)
    if record:
        states.append(dict(x=x.copy(), r=r.copy(), p=p.copy(), rho=float(rho)))
        return x, hist, states
    return x, hist
