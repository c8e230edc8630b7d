"""von Karman phase statistics (oracle, fp64).  Test infrastructure only.

Eq.53, with the reading G2 of DESIGN.md: the printed
"(r0/L0)^{5/6}" inside the bracket is a garble of (r/L0)^{5/6}, i.e.

    D_phi(r) = c2 (L0/r0)^{5/3} [ 1 - 2^{1/6}/Gamma(5/6) x^{5/6} K_{5/6}(x) ],  x = 2 pi r / L0,

which tends to 0 for r -> 0 because x^nu K_nu(x) -> 2^{nu-1} Gamma(nu).  The
prefactor is the exact constant c2 = 2 (24 Gamma(6/5)/5)^{5/6} Gamma(11/6) Gamma(5/6)
/ (2 pi^{8/3}) = 0.17262866 (the paper prints 0.17253).

Eq.45 (L559): Phi_phi(f) = 0.0229 r0^{-5/3} (f^2 + 1/L0^2)^{-11/6} (the printed 0.029
is a typo, reading G3); used here only to pin D_phi(inf) = 2 int Phi d^2f.
"""
import math

import numpy as np
from scipy.special import gamma, kv

C2 = 2.0 * (24.0 * gamma(6.0 / 5.0) / 5.0) ** (5.0 / 6.0) * gamma(11.0 / 6.0) * gamma(5.0 / 6.0) \
    / (2.0 * math.pi ** (8.0 / 3.0))
PSD_CONST = (24.0 * gamma(6.0 / 5.0) / 5.0) ** (5.0 / 6.0) * gamma(11.0 / 6.0) ** 2 \
    / (2.0 * math.pi ** (11.0 / 3.0))


def structure_function(r, r0: float, L0: float):
    """D_phi(r), Eq.53 (L619), r >= 0 in metres (array or scalar)."""
    r = np.asarray(r, dtype=np.float64)
    x = 2.0 * math.pi * r / L0
    out = np.zeros_like(x)
    nz = x > 0.0
    xs = x[nz]
    out[nz] = 1.0 - (2.0 ** (1.0 / 6.0) / gamma(5.0 / 6.0)) * xs ** (5.0 / 6.0) * kv(5.0 / 6.0, xs)
    return C2 * (L0 / r0) ** (5.0 / 3.0) * out


def structure_function_inf(r0: float, L0: float) -> float:
    """D_phi(r -> inf) = 2 * variance."""
    return C2 * (L0 / r0) ** (5.0 / 3.0)


def phase_covariance(r, r0: float, L0: float):
    """C_phi(r) = 1/2 D_phi(inf) - 1/2 D_phi(r)  (from Eq.49)."""
    return 0.5 * structure_function_inf(r0, L0) - 0.5 * structure_function(r, r0, L0)


def psd(f, r0: float, L0: float):
    """Phi_phi(|f|), Eq.45 (L559) with the corrected constant 0.0229 (exact value)."""
    f = np.asarray(f, dtype=np.float64)
    return PSD_CONST * r0 ** (-5.0 / 3.0) * (f * f + 1.0 / (L0 * L0)) ** (-11.0 / 6.0)
