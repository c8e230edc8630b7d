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

MINRES: `minres` below (the solver the paper keeps for the Toeplitz method, L426).
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


def minres(apply_A, b, n_iter: int, x0=None, dtype=np.float64, record=False):
    """Fixed-count MINRES (Paige & Saunders 1975), the solver the paper uses for the Toeplitz method (S2.G L337,
    L426 "MINRES and CG are used for the Toeplitz and sparse methods", Fig.13), un-preconditioned, cold start
    unless x0 is given (L428 warm start).  The paper prints no pseudo-code; this is the textbook form written out
    step by step: Lanczos tridiagonalisation of the symmetric A, QR of the tridiagonal by Givens rotations, update
    of the iterate along the directions w_k.

        r0 = b - A x0;  beta_1 = |r0|;  v_1 = r0 / beta_1;  v_0 = 0
        c_0 = -1, s_0 = 0, dbar_1 = 0, eps_1 = 0, phibar_0 = beta_1, w_0 = w_{-1} = 0
        for k = 1 .. n_iter:
            q       = A v_k
            alpha_k = v_k . q
            u       = q - alpha_k v_k - beta_k v_{k-1}
            beta_{k+1} = |u|
            delta_k   = c_{k-1} dbar_k + s_{k-1} alpha_k           (second super-diagonal entry after rotation k-1)
            gbar_k    = s_{k-1} dbar_k - c_{k-1} alpha_k
            eps_{k+1} = s_{k-1} beta_{k+1};   dbar_{k+1} = -c_{k-1} beta_{k+1}
            gamma_k = sqrt(gbar_k^2 + beta_{k+1}^2);  c_k = gbar_k / gamma_k;  s_k = beta_{k+1} / gamma_k
            phi_k = c_k phibar_{k-1};  phibar_k = s_k phibar_{k-1}
            w_k = (v_k - eps_k w_{k-2} - delta_k w_{k-1}) / gamma_k
            x_k = x_{k-1} + phi_k w_k
            v_{k+1} = u / beta_{k+1}

    x_k minimises |b - A x| over x0 + span{r0, A r0, .., A^{k-1} r0} and phibar_k is that minimum; the history is
    phibar_k, k = 0..n_iter.  Breakdown (beta_{k+1} = 0: the Krylov space is invariant, x_k is exact; or gamma_k = 0)
    freezes the iterate, like reading G16 for CG.
    Returns x, history[n_iter+1], and (if record) the per-iteration scalars and vectors.
    """
    b = np.asarray(b, dtype=dtype)
    if x0 is None:
        x = np.zeros_like(b)
        r0 = b.copy()
    else:
        x = np.asarray(x0, dtype=dtype).copy()
        r0 = (b - apply_A(x)).astype(dtype)
    beta = dtype(np.sqrt(dtype(r0 @ r0)))
    hist = [float(beta)]
    states = []
    v_old = np.zeros_like(b)
    v = (r0 / beta).astype(dtype) if beta > 0 else np.zeros_like(b)
    w1 = np.zeros_like(b)          # w_{k-1}
    w2 = np.zeros_like(b)          # w_{k-2}
    c, s = dtype(-1), dtype(0)
    dbar, eps, phibar = dtype(0), dtype(0), beta
    frozen = not (beta > 0)
    for _ in range(n_iter):
        if frozen:
            hist.append(float(phibar))
            if record:
                states.append(dict(frozen=True))
            continue
        q = np.asarray(apply_A(v), dtype=dtype)
        alpha = dtype(v @ q)
        u = (q - alpha * v - beta * v_old).astype(dtype)
        beta_next = dtype(np.sqrt(dtype(u @ u)))
        delta = dtype(c * dbar + s * alpha)
        gbar = dtype(s * dbar - c * alpha)
        eps_next = dtype(s * beta_next)
        dbar_next = dtype(-c * beta_next)
        gamma = dtype(np.sqrt(dtype(gbar * gbar + beta_next * beta_next)))
        if not (gamma > 0):
            frozen = True
            hist.append(float(phibar))
            if record:
                states.append(dict(frozen=True))
            continue
        c_new, s_new = dtype(gbar / gamma), dtype(beta_next / gamma)
        phi = dtype(c_new * phibar)
        phibar = dtype(s_new * phibar)
        w = ((v - eps * w2 - delta * w1) / gamma).astype(dtype)
        x = (x + phi * w).astype(dtype)
        if record:
            states.append(dict(alpha=float(alpha), beta=float(beta), beta_next=float(beta_next), gamma=float(gamma),
                               c=float(c_new), s=float(s_new), phi=float(phi), phibar=float(phibar),
                               v=v.copy(), w=w.copy(), x=x.copy(), frozen=False))
        w2, w1 = w1, w
        c, s, dbar, eps = c_new, s_new, dbar_next, eps_next
        hist.append(float(phibar))
        if beta_next > 0:
            v_old, v = v, (u / beta_next).astype(dtype)
            beta = beta_next
        else:
            frozen = True
    hist = np.asarray(hist)
    if record:
        return x, hist, states
    return x, hist
