"""Pins for oracle/vonkarman.py (Eq.53, Eq.45, Eq.49)."""
import math

import numpy as np
import pytest
from scipy import integrate, special

from oracle import vonkarman as vk

R0, L0 = 0.15, 25.0


def test_zero_and_infinity():
    assert vk.structure_function(0.0, R0, L0) == 0.0
    dinf = vk.structure_function_inf(R0, L0)
    assert abs(vk.structure_function(1e4, R0, L0) / dinf - 1) < 1e-12
    # monotone increasing
    r = np.linspace(0, 200, 4001)
    assert np.all(np.diff(vk.structure_function(r, R0, L0)) >= 0)


def test_constants_close_to_printed():
    rows = {}
    import os
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_closed_forms.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, val, tol, _ = [s.strip() for s in line.split("|", 3)]
            rows[name] = (float(val), float(tol))
    v, tol = rows["dphi_prefactor"]
    assert abs(vk.C2 / v - 1) < tol
    v, tol = rows["psd_constant"]
    assert abs(vk.PSD_CONST / v - 1) < tol


def test_kolmogorov_limit():
    # textbook: D(r) = 6.88 (r/r0)^{5/3} for r << L0; exact constant 2 (24/5 Gamma(6/5))^{5/6}
    c_kol = 2.0 * (24.0 / 5.0 * special.gamma(6.0 / 5.0)) ** (5.0 / 6.0)
    assert abs(c_kol - 6.8839) < 1e-3
    # next term of x^nu K_nu(x): D = c_kol (r/r0)^{5/3} [1 - 6 Gamma(11/6)/Gamma(1/6) (x/2)^{1/3} + O(x^2)]
    c1 = 6.0 * special.gamma(11.0 / 6.0) / special.gamma(1.0 / 6.0)
    big = 1e5
    for r in (0.05, 0.1, 0.5):
        d = float(vk.structure_function(r, R0, big))
        x = 2 * math.pi * r / big
        assert abs(d / (c_kol * (r / R0) ** (5.0 / 3.0) * (1 - c1 * (x / 2) ** (1.0 / 3.0))) - 1) < 2e-4


def test_variance_is_psd_integral():
    # D(inf)/2 = int Phi d^2f = 2 pi int_0^inf Phi(f) f df   (Wiener-Khinchin)
    val, _ = integrate.quad(lambda f: 2 * math.pi * f * vk.psd(f, R0, L0), 0, np.inf, limit=400)
    assert abs(val / (0.5 * vk.structure_function_inf(R0, L0)) - 1) < 1e-7


@pytest.mark.parametrize("r", [0.25, 0.5, 1.0, 5.0, 25.0])
def test_structure_function_is_hankel_of_psd(r):
    # D(r) = 2 int Phi(f) [1 - J0(2 pi f r)] 2 pi f df -- independent route to Eq.53
    def integrand(f):
        return 2.0 * vk.psd(f, R0, L0) * (1.0 - special.j0(2 * math.pi * f * r)) * 2 * math.pi * f
    # split the oscillatory tail: beyond f1 the "1" part is analytic, the J0 part is integrated with care
    f1 = 40.0 / r
    a, _ = integrate.quad(integrand, 0, f1, limit=2000)
    tail_one = 2.0 * 2 * math.pi * vk.PSD_CONST * R0 ** (-5 / 3) * \
        integrate.quad(lambda f: f * (f * f + 1 / L0 ** 2) ** (-11 / 6), f1, np.inf)[0]
    tail_j0, _ = integrate.quad(lambda f: 2.0 * vk.psd(f, R0, L0) * special.j0(2 * math.pi * f * r)
                                * 2 * math.pi * f, f1, 400.0 / r, limit=4000)
    ref = a + tail_one - tail_j0
    got = float(vk.structure_function(r, R0, L0))
    assert abs(got / ref - 1) < 2e-5


def test_bessel_agrees_with_second_library():
    # scipy's K_{5/6} against mpmath-free cross-check: integral representation
    # K_nu(x) = int_0^inf exp(-x cosh t) cosh(nu t) dt
    for x in (0.05, 0.1256637, 1.0, 6.0):
        ref, _ = integrate.quad(lambda t: math.exp(-x * math.cosh(t)) * math.cosh(5.0 / 6.0 * t), 0, 40)
        assert abs(special.kv(5.0 / 6.0, x) / ref - 1) < 1e-9


def test_small_argument_guard():
    # x^nu K_nu(x) -> 2^{nu-1} Gamma(nu): D -> 0 smoothly, no negative values
    r = np.array([1e-6, 1e-4, 1e-3])
    d = vk.structure_function(r, R0, L0)
    assert np.all(d >= 0) and d[0] < d[1] < d[2] < 1e-2
