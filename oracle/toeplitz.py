"""The paper's 2RBT (two-level recursive block Toeplitz) product, step by step (oracle).
Test infrastructure only.

S2.E: for an m^2 x n^2 2RBT matrix T with
T[(i,j),(i',j')] = g(i-i', j-j'), N1 = m+n-1:
  1. b = S_1 x,  b[mu1(i,j)] = x[i n + j],  mu1 = (m+n)(n-1) - i(m+n-1) - j     Eq.18-20
  2. b~ = F[b]   (1-D FFT of length N1^2)                                         Eq.21
  3. c~ = t~ . b~                                                                 Eq.22
  4. c = F^-1[c~]                                                                 Eq.23
  5. y[i m + j] = c[mu2(i,j)],  mu2 = (m+n)(m+n-1) - (i+1)(m+n-1) - (j+1)         Eq.24-26
Readings (G10): the printed ranges "(0 >= i,j >= n)" are 0 <= i,j < n (resp. < m);
the layout of t, never printed, must be t[u N1 + v] = g(m-1-u, m-1-v) for the steps to be exact.

The equivalent zero-padded 2-D form used on the GPU (any P >= m+n-1): K[(-l) mod P] = theta(l),
x in the top-left n x n corner, y = F2^-1[K~ . X~][0:m, 0:m], y[p] = sum_q theta(q - p) x[q].

Generators (L150, L265): theta_{(i,a),(j,b)}(l) = sum_k f_k cov_ab(gamma_k d l + h_k(alpha_j - alpha_i); d_k),
l in [-(n-1), n-1]^2; for the LGS phase-slope product (L193-197, reading G18)
xi'_{k,(j,b)}(l) = f_k cov_phi,b(d_k l + d_k[(n'-1)/2 - (n-1)/2] + h_k(alpha_j - beta); d_k),
l = q - p' in [-(n'-1), n-1]^2.
"""
import math

import numpy as np

from .covariance import cov_phase_slope, cov_slope_slope
from .geometry import ARCSEC, cone_factor


# ----------------------------------------------------------------------------- Eq.18-28
def mu1(i, j, m, n):
    return (m + n) * (n - 1) - i * (m + n - 1) - j          # Eq.20


def mu2(i, j, m, n):
    return (m + n) * (m + n - 1) - (i + 1) * (m + n - 1) - (j + 1)   # Eq.26


def t_vector(g, m, n):
    """Unique elements of T in the order the paper's steps need: t[u N1 + v] = g(m-1-u, m-1-v)."""
    N1 = m + n - 1
    t = np.zeros(N1 * N1)
    for u in range(N1):
        for v in range(N1):
            t[u * N1 + v] = g(m - 1 - u, m - 1 - v)
    return t


def rbt_mvm_paper(t, x, m, n):
    """y = T x by steps 1-5 above (1-D FFTs of length (m+n-1)^2)."""
    N1 = m + n - 1
    b = np.zeros(N1 * N1)
    for i in range(n):
        for j in range(n):
            b[mu1(i, j, m, n)] = x[i * n + j]                 # Eq.18-19
    c = np.fft.ifft(np.fft.fft(t) * np.fft.fft(b)).real      # Eq.21-23
    y = np.zeros(m * m)
    for i in range(m):
        for j in range(m):
            y[i * m + j] = c[mu2(i, j, m, n)]                 # Eq.24-25
    return y


def rbt_dense(g, m, n):
    """The explicit m^2 x n^2 matrix T[(i,j),(i',j')] = g(i-i', j-j')."""
    T = np.zeros((m * m, n * n))
    for i in range(m):
        for j in range(m):
            for ip in range(n):
                for jp in range(n):
                    T[i * m + j, ip * n + jp] = g(i - ip, j - jp)
    return T


def embed_generator(theta, n_in, n_out, P):
    """Circular embedding K[(-ly) mod P, (-lx) mod P] = theta(l) of a generator array
    theta[ly + (n_out-1), lx + (n_out-1)], l in [-(n_out-1), n_in-1]^2 (lag = input - output)."""
    if P < n_in + n_out - 1:
        raise ValueError("pad too small")
    K = np.zeros((P, P))
    for ly in range(-(n_out - 1), n_in):
        for lx in range(-(n_out - 1), n_in):
            K[(-ly) % P, (-lx) % P] = theta[ly + n_out - 1, lx + n_out - 1]
    return K


def rbt_mvm_fft2(theta, x_img, n_out, P):
    """y[p] = sum_q theta(q - p) x[q] through zero-padded 2-D FFTs of edge P."""
    n_in = x_img.shape[0]
    K = embed_generator(theta, n_in, n_out, P)
    X = np.zeros((P, P))
    X[:n_in, :n_in] = x_img
    Y = np.fft.ifft2(np.fft.fft2(K) * np.fft.fft2(X)).real
    return Y[:n_out, :n_out]


# ----------------------------------------------------------------------------- generators
def css_generators(n, d, wfs_dirs, h_gs, h, frac, r0, L0, model="hudgin", wfs_rows=None):
    """theta[i, a, j, b, ly+(n-1), lx+(n-1)]  (L150, L265).  wfs_rows: compute only the output WFSs i listed
    (the others stay zero) -- used to time a bounded sample of the ELT-size product; arithmetic unchanged."""
    N = len(wfs_dirs)
    L = 2 * n - 1
    lag = np.arange(-(n - 1), n)
    LX, LY = np.meshgrid(lag, lag, indexing="xy")
    lagv = np.stack([LX, LY], axis=-1).astype(np.float64)
    c = 1.0 / d
    th = np.zeros((N, 2, N, 2, L, L))
    for hk, fk in zip(h, frac):
        g = cone_factor(hk, h_gs)
        for i in (range(N) if wfs_rows is None else wfs_rows):
            for j in range(N):
                sh = hk * (np.asarray(wfs_dirs[j]) - np.asarray(wfs_dirs[i])) * ARCSEC
                delta = g * d * lagv + sh
                for a in range(2):
                    for b in range(2):
                        th[i, a, j, b] += fk * cov_slope_slope(delta, a, b, g * d, c, r0, L0, model)
    return th


def cos_generators(n, n_p, d, wfs_dirs, h_gs, beta, h, frac, r0, L0, model="hudgin"):
    """xi'[k, j, b, ly+(n'-1), lx+(n'-1)], lag l = q - p' (L193-197, reading G18)."""
    N = len(wfs_dirs)
    L = n_p + n - 1
    lag = np.arange(-(n_p - 1), n)
    LX, LY = np.meshgrid(lag, lag, indexing="xy")
    lagv = np.stack([LX, LY], axis=-1).astype(np.float64)
    c = 1.0 / d
    xi = np.zeros((len(h), N, 2, L, L))
    for k, (hk, fk) in enumerate(zip(h, frac)):
        g = cone_factor(hk, h_gs)
        dk = g * d
        off = dk * ((n_p - 1) / 2.0 - (n - 1) / 2.0)
        for j in range(N):
            sh = hk * (np.asarray(wfs_dirs[j]) - np.asarray(beta)) * ARCSEC
            delta = dk * lagv + off + sh
            for b in range(2):
                xi[k, j, b] = fk * cov_phase_slope(delta, b, dk, c, r0, L0, model)
    return xi


# ----------------------------------------------------------------------------- Eq.30 on the CPU
def css_spectra(theta, n, P):
    """theta~ for every block: rfft2 of the circular embedding (L265)."""
    N = theta.shape[0]
    out = np.zeros((N, 2, N, 2, P, P // 2 + 1), dtype=np.complex128)
    for i in range(N):
        for a in range(2):
            for j in range(N):
                for b in range(2):
                    out[i, a, j, b] = np.fft.rfft2(embed_generator(theta[i, a, j, b], n, n, P))
    return out


def css_mvm_fft(spec, x_full, n, P):
    """Sigma_ss x by Eq.30 (L267): 2N forward FFTs, 4N^2 spectral products summed per output
    channel, 2N inverse FFTs.  x_full: (N, 2, n, n) images on the full square grid."""
    N = spec.shape[0]
    X = np.zeros((N, 2, P, P))
    X[:, :, :n, :n] = x_full
    Xf = np.fft.rfft2(X)                                   # zeta~_q = F[S_1 zeta_q], once
    Yf = np.einsum("iajbyx,jbyx->iayx", spec, Xf)
    Y = np.fft.irfft2(Yf, s=(P, P))
    return Y[:, :, :n, :n]


# ----------------------------------------------------------------------------- closed forms
def ops_rbt(m, n, a=5.0):
    """(m+n-1)^2 [4a log(m+n-1) + 1] + m^2 + n^2   (L256); log = log2."""
    N1 = m + n - 1
    return N1 * N1 * (4 * a * math.log2(N1) + 1) + m * m + n * n


def ops_css(n, N, a=5.0):
    """4N{(2n-1)^2 [2a log(2n-1) + N] + n^2}   (L270)."""
    L = 2 * n - 1
    return 4 * N * (L * L * (2 * a * math.log2(L) + N) + n * n)


def reduction_css(n, N, a=5.0):
    """{(2n-1)^2[2a log(2n-1)+N]+n^2} N^-1 n^-4   (L270)."""
    return ops_css(n, N, a) / (4.0 * N * N * n ** 4)


def ops_cos_ngs(n, N, a=5.0):
    """2N[4n^2(2a log 2n + 1) + n^2] + 8n^2 log 2n + (n+1)^2   (L280)."""
    return 2 * N * (4 * n * n * (2 * a * math.log2(2 * n) + 1) + n * n) + 8 * n * n * math.log2(2 * n) \
        + (n + 1) ** 2


def ops_cos_lgs(n, n_p, N, K, a=5.0):
    """2(n'+n-1)^2[(2N+K) a log(n'+n-1) + N K] + 2N n^2 + 4K(n+1)^2   (L295)."""
    L = n_p + n - 1
    return 2 * L * L * ((2 * N + K) * a * math.log2(L) + N * K) + 2 * N * n * n + 4 * K * (n + 1) ** 2


def compression_css(n):
    return (2 * n - 1) ** 2 / n ** 4                                       # L150


def compression_cos_ngs(n):
    return 4.0 / (n + 1) ** 2                                              # L177


def compression_cos_lgs(n, n_p_list, N, K):
    """[sum_k (n'_k+n-1)^2](n+1)^-2 n^-2 + 2K N^-1 (n+1)^-2   (L197)."""
    return sum((npk + n - 1) ** 2 for npk in n_p_list) / ((n + 1) ** 2 * n ** 2) \
        + 2.0 * K / (N * (n + 1) ** 2)
