// host_kernels.cpp -- 2RBT generators of Sigma_ss and Sigma_phi-s and their spectra (row A0), fp64 on the host.
// Citations: PAPER.md L<line>.  Written from the paper; shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <limits>

#include "host_model.hpp"

namespace tomo {
namespace {
struct Tap { int u, v; double w; };

// Linear slope stencils on the phase, offsets in units of HALF the local subaperture width (App. A):
//   Hudgin-like Eq.47-48 (L584-594): s_x = c [phi(r + w/2 x^) - phi(r - w/2 x^)]
//   Fried       Eq.54-55 (L630-640): s_x = c/2 [phi(++) - phi(-+) - phi(--) + phi(+-)]
std::vector<Tap> stencil(int model, int comp) {
    if (model == TOMO_FRIED) {
        if (comp == 0) return {{+1, +1, +0.5}, {-1, +1, -0.5}, {-1, -1, -0.5}, {+1, -1, +0.5}};
        return {{+1, +1, +0.5}, {-1, +1, +0.5}, {-1, -1, -0.5}, {+1, -1, -0.5}};
    }
    if (comp == 0) return {{+1, 0, +1.0}, {-1, 0, -1.0}};
    return {{0, +1, +1.0}, {0, -1, -1.0}};
}

std::vector<Tap> pair_stencil(int model, int a, int b) {
    std::vector<Tap> out;
    for (const Tap &sa : stencil(model, a))
        for (const Tap &sb : stencil(model, b)) {
            const int u = sb.u - sa.u, v = sb.v - sa.v;
            bool found = false;
            for (Tap &t : out)
                if (t.u == u && t.v == v) { t.w += sa.w * sb.w; found = true; }
            if (!found) out.push_back({u, v, sa.w * sb.w});
        }
    out.erase(std::remove_if(out.begin(), out.end(), [](const Tap &t) { return t.w == 0.0; }), out.end());
    return out;
}

// D_phi on the half-step lattice {(hx, hy) * half + shift}: each value is needed by several lags and several
// component pairs (the +-d/2 arms of neighbouring lags coincide), so it is evaluated once.
struct Lattice {
    int lo, size;
    double half, sx, sy, r0, L0;
    std::vector<double> tab;
    Lattice(int lo_, int hi_, double half_, double sx_, double sy_, double r0_, double L0_)
        : lo(lo_), size(hi_ - lo_ + 1), half(half_), sx(sx_), sy(sy_), r0(r0_), L0(L0_),
          tab((size_t)size * size, std::numeric_limits<double>::quiet_NaN()) {}
    double get(int hx, int hy) {
        double &v = tab[(size_t)(hy - lo) * size + (hx - lo)];
        if (std::isnan(v)) v = structure_function(std::hypot(hx * half + sx, hy * half + sy), r0, L0);
        return v;
    }
};

// ---- FFT slope model (Eq.41-46; reading G29).  The slope is the gradient averaged over the subaperture; with
// H(f) = sinc(w f_x) sinc(w f_y) (Eq.44), the von Karman spectrum Phi (Eq.45, constant 0.0229: G3), slopes in rad/m and
// the cone compression gamma = w/d (L158):
//   cov(s_a(r), s_b(r + D))     = gamma^2 int (2 pi)^2 f_a f_b Phi H^2 cos(2 pi f.D) d^2f      (Eq.43)
//   cov(phi(r_p), s_b(r_p + D)) = -gamma  int  2 pi f_b      Phi H   sin(2 pi f.D) d^2f        (Eq.46)
// "computed by the FFT, accuracy depends on the sampling" (L572): Riemann sum over the grid of an FFT of edge NG with pixel
// w / kFftOver: f = p df, |p| < NG/2 (the unpaired Nyquist sample is left out), df = kFftOver / (NG w).  One inverse 2-D FFT
// gives the sum at every separation q (w / kFftOver) + shift; the lags of a generator are every kFftOver-th sample.
const int kFftOver = 4;
// Eq.45's constant, exact: (24 Gamma(6/5)/5)^(5/6) Gamma(11/6)^2 / (2 pi^(11/3)) = 0.022896 (the paper prints 0.029: G3)
const double kPsdConst = std::pow(24.0 * std::tgamma(6.0 / 5.0) / 5.0, 5.0 / 6.0) * std::tgamma(11.0 / 6.0) * std::tgamma(11.0 / 6.0) /
                         (2.0 * std::pow(M_PI, 11.0 / 3.0));

// Edge of the FFT grid (pixel w / kFftOver): a power of two >= 512 whose period NG w / kFftOver holds the largest separation
// the table is read at -- |lag| w PLUS the guide-star / target shift h_k d_alpha that enters as a phase ramp -- with at least
// one outer scale to the nearest alias (the table is the covariance periodised with that period; beyond L0 the slope
// covariances have decayed to < 1e-3 of the variance)
int fft_grid_edge(int max_lag, double w, double shx, double shy, double L0) {
    const double need = max_lag * w + std::max(std::fabs(shx), std::fabs(shy)) + L0;      // [m]
    int ng = 512;
    while (ng * w / kFftOver < need || kFftOver * max_lag >= ng / 2) ng *= 2;
    return std::min(ng, 8192);
}
double sinc_pi(double x) { return x == 0.0 ? 1.0 : std::sin(M_PI * x) / (M_PI * x); }

// tab[(qy mod NG) NG + (qx mod NG)] = sum_p weight(fx, fy) exp(2 pi i f.(q w/kFftOver + shift)); kind 0/1/2 = Sigma_ss xx / yy / xy
// (real part), 3/4 = Sigma_phi-s x / y (imaginary part)
void fft_model_table(int NG, double w, double gam, double r0, double L0, double shx, double shy, int kind,
                     std::vector<std::complex<double>> &tab) {
    typedef std::complex<double> cd;
    const double df = kFftOver / (NG * w);
    tab.assign((size_t)NG * NG, cd(0, 0));
    for (int py = -(NG / 2 - 1); py < NG / 2; ++py)
        for (int px = -(NG / 2 - 1); px < NG / 2; ++px) {
            const double fx = px * df, fy = py * df;
            const double H = sinc_pi(w * fx) * sinc_pi(w * fy);
            const double phi = kPsdConst * std::pow(r0, -5.0 / 3.0) * std::pow(fx * fx + fy * fy + 1.0 / (L0 * L0), -11.0 / 6.0);
            double wt;
            if (kind < 3) {
                const double fa = (kind == 1) ? fy : fx, fb = (kind == 0) ? fx : fy;
                wt = gam * gam * 4.0 * M_PI * M_PI * fa * fb * phi * H * H * df * df;
            } else {
                wt = -gam * 2.0 * M_PI * (kind == 3 ? fx : fy) * phi * H * df * df;
            }
            const double ph = 2.0 * M_PI * (fx * shx + fy * shy);
            tab[(size_t)((py + NG) % NG) * NG + ((px + NG) % NG)] = wt * cd(std::cos(ph), std::sin(ph));
        }
    for (int y = 0; y < NG; ++y) host_fft(&tab[(size_t)y * NG], NG, 1, true);       // inverse: exp(+2 pi i p q / NG), unscaled
    for (int x = 0; x < NG; ++x) host_fft(&tab[x], NG, NG, true);
}
}  // namespace

// 1/2 [theta_x0x0(0) + theta_y0y0(0)]: the model slope variance the noise level is quoted against (reading G15)
double model_slope_variance(const HostModel &m) {
    double v = 0.0;
    const double c = 1.0 / m.d;
    if (m.slope_model == TOMO_FFTMODEL) {
        for (int k = 0; k < m.K; ++k) {
            const double w = m.gamma[k] * m.d;
            const int NG = fft_grid_edge(m.n_p, w, 0.0, 0.0, m.L0);
            const double df = kFftOver / (NG * w);
            double s = 0.0;
            for (int py = -(NG / 2 - 1); py < NG / 2; ++py)
                for (int px = -(NG / 2 - 1); px < NG / 2; ++px) {
                    const double fx = px * df, fy = py * df, H = sinc_pi(w * fx) * sinc_pi(w * fy);
                    const double phi = kPsdConst * std::pow(m.r0, -5.0 / 3.0) * std::pow(fx * fx + fy * fy + 1.0 / (m.L0 * m.L0), -11.0 / 6.0);
                    s += 4.0 * M_PI * M_PI * (fx * fx + fy * fy) * phi * H * H * df * df;
                }
            v += m.frac[k] * m.gamma[k] * m.gamma[k] * s;
        }
        return 0.5 * v;
    }
    for (int k = 0; k < m.K; ++k) {
        const double w = m.gamma[k] * m.d;
        Lattice lat(-2, 2, 0.5 * w, 0.0, 0.0, m.r0, m.L0);
        for (int a = 0; a < 2; ++a) {
            double s = 0.0;
            for (const Tap &t : pair_stencil(m.slope_model, a, a)) s += t.w * lat.get(t.u, t.v);
            v += m.frac[k] * (-0.5 * c * c) * s;
        }
    }
    return 0.5 * v;
}

// ------------------------------------------------------------------------------------------------ Sigma_ss
// theta[(i,a),(j,b)](l) = sum_k f_k cov_ab(gamma_k d l + h_k (alpha_j - alpha_i); d_k)        (L150, L158, L265)
// cov_ab(Delta; w)      = -1/2 c^2 sum_{m,m'} w_m w'_m' D_phi(|Delta + o'_m' - o_m|), c = 1/d  (Eq.49;
//                         Eq.50-52 are the Hudgin special cases, Eq.51's last sign corrected -- reading G4)
void build_css_generators(const HostModel &m, std::vector<double> &gen) {
    const int n = m.n, N = m.n_wfs, C = m.C, L = 2 * n - 1, K = m.K;
    const size_t LL = (size_t)L * L;
    gen.assign((size_t)C * C * LL, 0.0);
    const double c = 1.0 / m.d;
    std::vector<Tap> st[2][2];
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) st[a][b] = pair_stencil(m.slope_model, a, b);
    // distinct WFS pairs: (0,0) stands for every i == j (zero shift), plus all i < j
    std::vector<std::pair<int, int>> pairs;
    pairs.push_back({0, 0});
    for (int i = 0; i < N; ++i)
        for (int j = i + 1; j < N; ++j) pairs.push_back({i, j});
    std::vector<double> tmp((size_t)K * 4 * LL);
    for (const auto &pr : pairs) {
        const int i = pr.first, j = pr.second;
#pragma omp parallel for schedule(dynamic)
        for (int k = 0; k < K; ++k) {
            const double w = m.gamma[k] * m.d;
            const double shx = m.h[k] * (m.ax[j] - m.ax[i]), shy = m.h[k] * (m.ay[j] - m.ay[i]);
            if (m.slope_model == TOMO_FFTMODEL) {
                const int NG = fft_grid_edge(n, w, shx, shy, m.L0);
                std::vector<std::complex<double>> tab;
                for (int a = 0; a < 2; ++a)
                    for (int b = a; b < 2; ++b) {
                        fft_model_table(NG, w, m.gamma[k], m.r0, m.L0, shx, shy, a == b ? a : 2, tab);
                        for (int ly = -(n - 1); ly < n; ++ly)
                            for (int lx = -(n - 1); lx < n; ++lx) {
                                const double val = m.frac[k] * tab[(size_t)((kFftOver * ly + NG) % NG) * NG + ((kFftOver * lx + NG) % NG)].real();
                                tmp[((size_t)k * 4 + a * 2 + b) * LL + (size_t)(ly + n - 1) * L + (lx + n - 1)] = val;
                                if (a != b) tmp[((size_t)k * 4 + b * 2 + a) * LL + (size_t)(ly + n - 1) * L + (lx + n - 1)] = val;
                            }
                    }
                continue;
            }
            Lattice lat(-2 * n, 2 * n, 0.5 * w, shx, shy, m.r0, m.L0);
            const double scale = m.frac[k] * (-0.5 * c * c);
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < 2; ++b) {
                    double *o = &tmp[((size_t)k * 4 + a * 2 + b) * LL];
                    for (int ly = -(n - 1); ly < n; ++ly)
                        for (int lx = -(n - 1); lx < n; ++lx) {
                            double s = 0.0;
                            for (const Tap &t : st[a][b]) s += t.w * lat.get(2 * lx + t.u, 2 * ly + t.v);
                            o[(size_t)(ly + n - 1) * L + (lx + n - 1)] = scale * s;
                        }
                }
        }
        // layer sum in a fixed order (deterministic), then place the block(s)
        std::vector<double> acc(4 * LL, 0.0);
#pragma omp parallel for schedule(static)
        for (long e = 0; e < (long)(4 * LL); ++e) {
            double s = 0.0;
            for (int k = 0; k < K; ++k) s += tmp[(size_t)k * 4 * LL + e];
            acc[e] = s;
        }
        auto place = [&](int wi, int wj) {
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < 2; ++b) {
                    const int co = 2 * wi + a, ci = 2 * wj + b;
                    double *dst = &gen[((size_t)co * C + ci) * LL];
                    double *dstT = &gen[((size_t)ci * C + co) * LL];
                    const double *src = &acc[(size_t)(a * 2 + b) * LL];
                    for (size_t e = 0; e < LL; ++e) dst[e] = src[e];
                    if (wi != wj)   // theta_{(j,b),(i,a)}(l) = theta_{(i,a),(j,b)}(-l)
                        for (size_t e = 0; e < LL; ++e) dstT[LL - 1 - e] = src[e];
                }
        };
        if (i == j) for (int w = 0; w < N; ++w) place(w, w);
        else place(i, j);
    }
}

// ------------------------------------------------------------------------------------------------ low-order NGS path
// Reading G30 (the paper is silent: L321, L412).  Sensor m and target t are described by the aperture-mean slope pair in
// their direction (NGS / infinity: no cone compression).  With c(l) the autocorrelation count of the subaperture mask,
//   cov(mean_a(u), mean_b(v)) = 1/n_vs^2 sum_l c(l) sum_k f_k cov_ab(d l + h_k (v - u); d)
// (the same cov_ab as Sigma_ss, Eq.49).  R_lo = C_tau,g (C_gg + sigma2_lo I)^-1 by Cholesky (Eq.5).
int build_lo_estimator(const HostModel &m, const std::vector<double> &ux, const std::vector<double> &uy, int n_lo,
                       double sigma2_lo, std::vector<double> &R, std::vector<double> &Cm) {
    const int n = m.n, L = 2 * n - 1, K = m.K, M = (int)ux.size(), T = M - n_lo, n_g = 2 * n_lo;
    const size_t LL = (size_t)L * L;
    std::vector<double> cnt(LL, 0.0);
    for (int q = 0; q < m.nv; ++q)
        for (int p = 0; p < m.nv; ++p) cnt[(size_t)(m.iy[p] - m.iy[q] + n - 1) * L + (m.ix[p] - m.ix[q] + n - 1)] += 1.0;
    std::vector<Tap> st[2][2];
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) st[a][b] = pair_stencil(m.slope_model, a, b);
    const double c = 1.0 / m.d, inv = 1.0 / ((double)m.nv * m.nv);
    Cm.assign((size_t)4 * M * M, 0.0);
    std::vector<std::pair<int, int>> pairs;
    for (int i = 0; i < M; ++i)
        for (int j = i; j < M; ++j) pairs.push_back({i, j});
#pragma omp parallel for schedule(dynamic)
    for (int e = 0; e < (int)pairs.size(); ++e) {
        const int i = pairs[e].first, j = pairs[e].second;
        double acc[2][2] = {{0, 0}, {0, 0}};
        for (int k = 0; k < K; ++k) {
            Lattice lat(-2 * n, 2 * n, 0.5 * m.d, m.h[k] * (ux[j] - ux[i]), m.h[k] * (uy[j] - uy[i]), m.r0, m.L0);
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < 2; ++b) {
                    double s = 0.0;
                    for (int ly = -(n - 1); ly < n; ++ly)
                        for (int lx = -(n - 1); lx < n; ++lx) {
                            const double w = cnt[(size_t)(ly + n - 1) * L + (lx + n - 1)];
                            if (w == 0.0) continue;
                            double v = 0.0;
                            for (const Tap &t : st[a][b]) v += t.w * lat.get(2 * lx + t.u, 2 * ly + t.v);
                            s += w * v;
                        }
                    acc[a][b] += m.frac[k] * (-0.5 * c * c) * s * inv;
                }
        }
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b) {
                Cm[(size_t)(2 * i + a) * 2 * M + (2 * j + b)] = acc[a][b];
                Cm[(size_t)(2 * j + b) * 2 * M + (2 * i + a)] = acc[a][b];
            }
    }
    // Cholesky of A = C_gg + sigma2_lo I, then R^T = A^-1 C_g,tau column by column
    std::vector<double> A((size_t)n_g * n_g);
    for (int r = 0; r < n_g; ++r)
        for (int q = 0; q < n_g; ++q) A[(size_t)r * n_g + q] = Cm[(size_t)r * 2 * M + q] + (r == q ? sigma2_lo : 0.0);
    for (int r = 0; r < n_g; ++r)
        for (int q = 0; q <= r; ++q) {
            double s = A[(size_t)r * n_g + q];
            for (int p = 0; p < q; ++p) s -= A[(size_t)r * n_g + p] * A[(size_t)q * n_g + p];
            if (r == q) {
                if (!(s > 0.0)) return TOMO_EINVAL;
                A[(size_t)r * n_g + r] = std::sqrt(s);
            } else {
                A[(size_t)r * n_g + q] = s / A[(size_t)q * n_g + q];
            }
        }
    R.assign((size_t)2 * T * n_g, 0.0);
    std::vector<double> y(n_g);
    for (int row = 0; row < 2 * T; ++row) {
        for (int r = 0; r < n_g; ++r) {
            double s = Cm[(size_t)(n_g + row) * 2 * M + r];
            for (int p = 0; p < r; ++p) s -= A[(size_t)r * n_g + p] * y[p];
            y[r] = s / A[(size_t)r * n_g + r];
        }
        for (int r = n_g - 1; r >= 0; --r) {
            double s = y[r];
            for (int p = r + 1; p < n_g; ++p) s -= A[(size_t)p * n_g + r] * R[(size_t)row * n_g + p];
            R[(size_t)row * n_g + r] = s / A[(size_t)r * n_g + r];
        }
    }
    return TOMO_OK;
}

// ------------------------------------------------------------------------------------------------ Sigma_phi-s
// xi'[k,(j,b)](l) = f_k cov_phi,b(d_k l + d_k[(n'-1)/2 - (n-1)/2] + h_k (alpha_j - beta); d_k),  l = q - p'
// cov_phi,b(Delta; w) = -1/2 c sum_m' w'_m' D_phi(|Delta + o'_m'|)            (Eq.52; L179-197; reading G18)
// NGS systems: gamma_k = 1, n' = n+1, and the layers are summed into one table (Eq.15, Eq.31).
void build_cos_generators(const HostModel &m, int target, std::vector<double> &gen) {
    const int n = m.n, np = m.n_p, N = m.n_wfs, C = m.C, Los = np + n - 1, K = m.K;
    const size_t LL = (size_t)Los * Los;
    gen.assign((size_t)m.Kp * C * LL, 0.0);
    const double c = 1.0 / m.d;
    std::vector<Tap> st[2] = {stencil(m.slope_model, 0), stencil(m.slope_model, 1)};
    std::vector<double> tmp;
    if (!m.per_layer()) tmp.assign((size_t)K * C * LL, 0.0);
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int k = 0; k < K; ++k)
        for (int j = 0; j < N; ++j) {
            const double w = m.gamma[k] * m.d;
            const double off = w * ((np - 1) / 2.0 - (n - 1) / 2.0);
            const double shx = off + m.h[k] * (m.ax[j] - m.bx[target]);
            const double shy = off + m.h[k] * (m.ay[j] - m.by[target]);
            if (m.slope_model == TOMO_FFTMODEL) {
                const int NG = fft_grid_edge(m.n_p, w, shx, shy, m.L0);
                std::vector<std::complex<double>> tab;
                for (int b = 0; b < 2; ++b) {
                    fft_model_table(NG, w, m.gamma[k], m.r0, m.L0, shx, shy, 3 + b, tab);
                    double *o = m.per_layer() ? &gen[((size_t)k * C + 2 * j + b) * LL] : &tmp[((size_t)k * C + 2 * j + b) * LL];
                    for (int ly = -(np - 1); ly < n; ++ly)
                        for (int lx = -(np - 1); lx < n; ++lx)
                            o[(size_t)(ly + np - 1) * Los + (lx + np - 1)] =
                                m.frac[k] * tab[(size_t)((kFftOver * ly + NG) % NG) * NG + ((kFftOver * lx + NG) % NG)].imag();
                }
                continue;
            }
            Lattice lat(-2 * np, 2 * n, 0.5 * w, shx, shy, m.r0, m.L0);
            const double scale = m.frac[k] * (-0.5 * c);
            for (int b = 0; b < 2; ++b) {
                double *o = m.per_layer() ? &gen[((size_t)k * C + 2 * j + b) * LL] : &tmp[((size_t)k * C + 2 * j + b) * LL];
                for (int ly = -(np - 1); ly < n; ++ly)
                    for (int lx = -(np - 1); lx < n; ++lx) {
                        double s = 0.0;
                        for (const Tap &t : st[b]) s += t.w * lat.get(2 * lx + t.u, 2 * ly + t.v);
                        o[(size_t)(ly + np - 1) * Los + (lx + np - 1)] = scale * s;
                    }
            }
        }
    if (!m.per_layer()) {
#pragma omp parallel for schedule(static)
        for (long e = 0; e < (long)((size_t)C * LL); ++e) {
            double s = 0.0;
            for (int k = 0; k < K; ++k) s += tmp[(size_t)k * C * LL + e];
            gen[e] = s;
        }
    }
}

// ------------------------------------------------------------------------------------------------ host FFT
// Stockham autosort, radices 2/3/4/5 by direct small DFTs; exact enough (fp64) and only used at plan build.
void host_fft(std::complex<double> *x, int n, int stride, bool inverse) {
    typedef std::complex<double> cd;
    std::vector<cd> a(n), b(n);
    for (int i = 0; i < n; ++i) a[i] = x[(size_t)i * stride];
    std::vector<cd> tw(n);
    const double sgn = inverse ? +1.0 : -1.0;
    for (int t = 0; t < n; ++t) tw[t] = cd(std::cos(2.0 * M_PI * t / n), sgn * std::sin(2.0 * M_PI * t / n));
    int ncur = n, s = 1;
    cd *src = a.data(), *dst = b.data();
    while (ncur > 1) {
        int r = (ncur % 4 == 0) ? 4 : (ncur % 2 == 0) ? 2 : (ncur % 3 == 0) ? 3 : 5;
        const int mm = ncur / r;
        for (int p = 0; p < mm; ++p)
            for (int q = 0; q < s; ++q) {
                cd in[5];
                for (int j = 0; j < r; ++j) in[j] = src[q + s * (p + mm * j)];
                for (int k = 0; k < r; ++k) {
                    cd acc(0, 0);
                    for (int j = 0; j < r; ++j) acc += in[j] * tw[(size_t)((j * k) % r) * (n / r)];
                    dst[q + s * (r * p + k)] = acc * tw[(size_t)p * k * s];
                }
            }
        ncur = mm; s *= r;
        std::swap(src, dst);
    }
    for (int i = 0; i < n; ++i) x[(size_t)i * stride] = src[i];
}

// K[(-l) mod P] = g(l); out = rfft2(K)/P^2 stored [kx][ky]   (L207, L265; readings G10, G24)
void generator_spectrum(const double *g, int n_out, int n_in, int P, std::complex<double> *out) {
    typedef std::complex<double> cd;
    const int Lg = n_out + n_in - 1, Ph = P / 2 + 1;
    std::vector<cd> img((size_t)P * P, cd(0, 0));
    for (int ly = -(n_out - 1); ly < n_in; ++ly)
        for (int lx = -(n_out - 1); lx < n_in; ++lx)
            img[(size_t)(((-ly) % P + P) % P) * P + (((-lx) % P + P) % P)] = g[(size_t)(ly + n_out - 1) * Lg + (lx + n_out - 1)];
    for (int y = 0; y < P; ++y) host_fft(&img[(size_t)y * P], P, 1, false);     // along x
    const double sc = 1.0 / ((double)P * P);
    for (int kx = 0; kx < Ph; ++kx) {
        host_fft(&img[kx], P, P, false);                                          // along y
        for (int ky = 0; ky < P; ++ky) out[(size_t)kx * P + ky] = img[(size_t)ky * P + kx] * sc;
    }
}

}  // namespace tomo
