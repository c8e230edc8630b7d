"""Assemble a TomoConfig into the oracle's operator, right-hand side and projection.
Test infrastructure only.

Dense mode (tiny / mid): every matrix explicit, built from positions (covariance.py):
    A   = M_s (W_s Sigma_ss W_s^T + Sigma_eta) M_s^T      Eq.34 (L311), L329
    b   = M_s s
    phi = M_phi W_phi Sigma_{phi s} W_s^T M_s^T zeta       Eq.35 (L313), L329
with Sigma_{phi s} the direct covariance for NGS systems (Eq.15) and the paper's
interpolated form sum_k I'_k Xi'_k (Eq.17) for LGS systems.

Matrix-free mode (ELT sizes, 51 648^2 fp64 = 21 GB dense): the same operator with the
Sigma_ss product done entry by entry from the generators (directsum.c), no FFT.

Noise (reading G15): Sigma_eta = sigma^2 I, sigma^2 = noise_frac * 1/2 [theta_x0x0(0) + theta_y0y0(0)]; optionally the
2 x 2 block-diagonal Sigma_eta of elongated LGS spots (L331-333), given entry by entry.
"""
import math

import numpy as np

from . import covariance as cov
from . import geometry as geo
from . import projectors as prj
from . import solver
from . import toeplitz as tz


class OracleSystem:
    def __init__(self, cfg, model: str = "hudgin", dense: bool = True, build_cos: bool = True, noise_blocks=None):
        """noise_blocks = (sxx, syy, sxy), each [n_wfs][n_vs]: Sigma_eta with one 2 x 2 block [[sxx, sxy], [sxy, syy]] per
        subaperture coupling its x- and y-slope (elongated LGS spots, L331-333); None = sigma^2 I (G15)."""
        if noise_blocks is not None and not dense:
            raise ValueError("2 x 2 noise blocks are only assembled in dense mode")
        self.cfg = cfg
        self.model = model
        n, d = cfg.n, cfg.d
        self.n, self.d = n, d
        self.N = cfg.n_wfs
        self.smask = geo.subap_mask(n, cfg.D, cfg.obstruction)
        self.pmask = geo.phase_mask(self.smask)
        self.sub_idx = np.flatnonzero(self.smask.ravel())
        self.ph_idx = np.flatnonzero(self.pmask.ravel())
        self.nv = self.sub_idx.size
        self.nvp = self.ph_idx.size
        self.centres = geo.subap_centres(n, d)[self.sub_idx]
        self.phase_pts = geo.phase_points(n, d)[self.ph_idx]
        self.ix = (self.sub_idx % n).astype(np.int32)
        self.iy = (self.sub_idx // n).astype(np.int32)
        self.dirs = [(w.ax, w.ay) for w in cfg.wfs]
        self.hgs = [w.h_gs for w in cfg.wfs]
        if len(set(self.hgs)) != 1:
            raise ValueError("high-order WFSs must share one guide-star altitude (L158)")
        self.h_gs = self.hgs[0]
        self.is_lgs = not math.isinf(self.h_gs)
        self.n_remove = [w.n_remove for w in cfg.wfs]
        self.n_remove_phase = max(self.n_remove) if self.is_lgs else 0
        self.Ns = 2 * self.N * self.nv
        # noise variance from the model variance of WFS 0 (G15)
        z = np.zeros((1, 2))
        v = 0.0
        for hk, fk in zip(cfg.h, cfg.frac):
            g = geo.cone_factor(hk, self.h_gs)
            for a in range(2):
                v += fk * cov.cov_slope_slope(z, a, a, g * d, 1.0 / d, cfg.r0, cfg.L0, model)[0]
        self.slope_var = 0.5 * v
        self.sigma2 = cfg.noise_frac * self.slope_var
        gam_min = min(geo.cone_factor(hk, self.h_gs) for hk in cfg.h)
        self.n_p = geo.n_prime(n, gam_min)
        self.Ms = prj.slope_projector(self.centres, self.n_remove) if dense or self.Ns <= 6000 else None
        self.Mphi = prj.phase_projector(self.phase_pts, self.n_remove_phase)
        self.dense = dense
        self.Css = None
        self.A = None
        self.theta = None
        self.Cos = None
        if dense:
            self.Css = cov.dense_css(self.centres, d, self.dirs, self.hgs, cfg.h, cfg.frac,
                                     cfg.r0, cfg.L0, model)
            self.Cnn = self.sigma2 * np.eye(self.Ns)
            if noise_blocks is not None:
                sxx, syy, sxy = (np.asarray(a, dtype=np.float64).reshape(self.N, self.nv) for a in noise_blocks)
                self.Cnn = np.zeros((self.Ns, self.Ns))
                for i in range(self.N):
                    for q in range(self.nv):
                        ex, ey = (2 * i) * self.nv + q, (2 * i + 1) * self.nv + q     # [wfs][x then y][subaperture] (Eq.29)
                        self.Cnn[ex, ex], self.Cnn[ey, ey] = sxx[i, q], syy[i, q]
                        self.Cnn[ex, ey] = self.Cnn[ey, ex] = sxy[i, q]
            self.A = self.Ms @ (self.Css + self.Cnn) @ self.Ms.T
            if build_cos:
                self.Cos = [self._dense_cos(beta) for beta in cfg.targets]

    # ------------------------------------------------------------------ pieces
    def _dense_cos(self, beta):
        c = self.cfg
        if self.is_lgs:
            return cov.dense_cos_interpolated(self.phase_pts, self.centres, self.d, self.dirs, self.h_gs,
                                              beta, c.h, c.frac, c.r0, c.L0, self.n_p, self.model)
        return cov.dense_cos_direct(self.phase_pts, self.centres, self.d, self.dirs, self.hgs, beta,
                                    c.h, c.frac, c.r0, c.L0, self.model)

    def dense_cos_direct(self, beta):
        c = self.cfg
        return cov.dense_cos_direct(self.phase_pts, self.centres, self.d, self.dirs, self.hgs, beta,
                                    c.h, c.frac, c.r0, c.L0, self.model)

    def project_slopes(self, v):
        """M_s v, mode by mode (the same Z of projectors.py, applied per WFS)."""
        if self.Ms is not None:
            return self.Ms @ v
        out = np.array(v, dtype=np.float64).reshape(self.N, 2 * self.nv)
        for i, nr in enumerate(self.n_remove):
            Z = prj.slope_modes(self.centres, nr)
            if Z.shape[1]:
                out[i] -= Z @ (np.linalg.pinv(Z) @ out[i])
        return out.ravel()

    def generators(self):
        if self.theta is None:
            c = self.cfg
            self.theta = tz.css_generators(self.n, self.d, self.dirs, self.h_gs, c.h, c.frac,
                                           c.r0, c.L0, self.model)
        return self.theta

    # ------------------------------------------------------------------ operator
    def apply_A(self, v):
        """A v with A = M_s (W Sigma_ss W^T + sigma^2 I) M_s^T."""
        if self.dense:
            return self.A @ v
        from . import directsum
        u = self.project_slopes(v)
        q = directsum.css_mvm(self.generators(), self.ix, self.iy, u) + self.sigma2 * u
        return self.project_slopes(q)

    def css_rows_explicit(self, rows):
        """Selected rows of W_s Sigma_ss W_s^T built from POSITIONS exactly as covariance.dense_css does (Eq.14,
        L158): the row-sampled check that pins the generator / direct-sum route at sizes where the dense matrix does
        not fit.  rows: flat indices (i, a, q) -> (i*2 + a)*nv + q.  Returns (len(rows), Ns)."""
        c = self.cfg
        out = np.zeros((len(rows), self.N, 2, self.nv))
        for t, row in enumerate(rows):
            ch, q = divmod(int(row), self.nv)
            i, a = divmod(ch, 2)
            for hk, fk in zip(c.h, c.frac):
                g = geo.cone_factor(hk, self.h_gs)
                pos_i = g * self.centres[q] + hk * np.asarray(self.dirs[i]) * geo.ARCSEC
                for j in range(self.N):
                    pos_j = g * self.centres + hk * np.asarray(self.dirs[j]) * geo.ARCSEC
                    delta = pos_j - pos_i[None, :]
                    for b in range(2):
                        out[t, j, b] += fk * cov.cov_slope_slope(delta, a, b, g * self.d, 1.0 / self.d, c.r0, c.L0,
                                                                 self.model)
        return out.reshape(len(rows), self.Ns)

    def css_unprojected(self, u):
        """W_s Sigma_ss W_s^T u without noise and projectors (dense or direct-sum)."""
        if self.dense:
            return self.Css @ u
        from . import directsum
        return directsum.css_mvm(self.generators(), self.ix, self.iy, np.asarray(u, dtype=np.float64))

    def rhs(self, slopes):
        return self.project_slopes(np.asarray(slopes, dtype=np.float64))

    def solve_direct(self, slopes):
        singular = any(nr > 0 for nr in self.n_remove)
        return solver.direct_solve(self.A, self.rhs(slopes), singular)

    def solve_cg(self, slopes, n_iter, x0=None, record=False, dtype=np.float64):
        b = self.rhs(slopes)
        if dtype == np.float64:
            f = self.apply_A
        else:
            A32 = self.A.astype(dtype)
            f = lambda v: A32 @ v          # noqa: E731  fp32 emulation of the same algorithm
        return solver.cg(f, b, n_iter, x0=x0, dtype=dtype, record=record)

    def solve_minres(self, slopes, n_iter, x0=None, record=False, dtype=np.float64):
        """Fixed-count MINRES on the same system (the paper's solver for the Toeplitz method, L426)."""
        b = self.rhs(slopes)
        if dtype == np.float64:
            f = self.apply_A
        else:
            A32 = self.A.astype(dtype)
            f = lambda v: A32 @ v          # noqa: E731  fp32 emulation of the same algorithm
        return solver.minres(f, b, n_iter, x0=x0, dtype=dtype, record=record)

    # ------------------------------------------------------------------ projection, Eq.13/35
    def reconstruct(self, zeta, target: int = 0):
        """phi_hat = M_phi W_phi Sigma_{phi s} W_s^T M_s^T zeta over the valid phase points."""
        z = self.project_slopes(np.asarray(zeta, dtype=np.float64))
        if self.Cos is not None:
            return self.Mphi @ (self.Cos[target] @ z)
        return self.Mphi @ self.cos_matrix_free(z, target)

    def cos_matrix_free(self, z, target: int = 0):
        """sum_k I'_k Xi'_k z (Eq.32 L290 without FFTs) from the per-layer generators, entry by
        entry (directsum.c), then the 4-tap bilinear I'_k."""
        from . import directsum
        c = self.cfg
        beta = c.targets[target]
        out = np.zeros(self.nvp)
        for k, (hk, fk) in enumerate(zip(c.h, c.frac)):
            xi = tz.cos_generators(self.n, self.n_p, self.d, self.dirs, self.h_gs, beta,
                                   [hk], [fk], c.r0, c.L0, self.model)[0]
            g = directsum.cos_layer(xi, self.n, self.n_p, self.ix, self.iy, z)
            dk = geo.cone_factor(hk, self.h_gs) * self.d
            t = self.phase_pts / dk + (self.n_p - 1) / 2.0
            i0x = np.clip(np.floor(t[:, 0] + 1e-12).astype(int), 0, self.n_p - 2)
            i0y = np.clip(np.floor(t[:, 1] + 1e-12).astype(int), 0, self.n_p - 2)
            wx = t[:, 0] - i0x
            wy = t[:, 1] - i0y
            out += (1 - wx) * (1 - wy) * g[i0y, i0x] + wx * (1 - wy) * g[i0y, i0x + 1] \
                + (1 - wx) * wy * g[i0y + 1, i0x] + wx * wy * g[i0y + 1, i0x + 1]
        return out
