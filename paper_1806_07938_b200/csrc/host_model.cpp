// host_model.cpp -- see host_model.hpp.  fp64 throughout; OpenMP over independent tables.
#include "host_model.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>

namespace tomo {

// ------------------------------------------------------------------------------------------------ sizes
bool is_5smooth(int v) {
    if (v < 1) return false;
    for (int f : {2, 3, 5})
        while (v % f == 0) v /= f;
    return v == 1;
}

int next_fft_size(int v) {
    int p = std::max(v, 2);
    while (!(p % 2 == 0 && is_5smooth(p))) ++p;
    return p;
}

// ------------------------------------------------------------------------------------------------ Eq.53
// D_phi(r) = c2 (L0/r0)^{5/3} [1 - 2^{1/6}/Gamma(5/6) x^{5/6} K_{5/6}(x)], x = 2 pi r/L0   (L619; reading G2:
// the printed (r0/L0)^{5/6} inside the bracket is (r/L0)^{5/6}, and c2 is the exact constant, printed 0.17253).
double structure_function(double r, double r0, double L0) {
    static const double c2 = 2.0 * std::pow(24.0 * std::tgamma(6.0 / 5.0) / 5.0, 5.0 / 6.0) * std::tgamma(11.0 / 6.0) *
                             std::tgamma(5.0 / 6.0) / (2.0 * std::pow(M_PI, 8.0 / 3.0));
    static const double kc = std::pow(2.0, 1.0 / 6.0) / std::tgamma(5.0 / 6.0);
    const double amp = c2 * std::pow(L0 / r0, 5.0 / 3.0);
    if (!(r > 0.0)) return 0.0;
    const double x = 2.0 * M_PI * r / L0;
    if (x < 1e-4) {
        // 1 - kc x^nu K_nu(x) cancels for tiny x (G23): leading term of the series,
        // x^nu K_nu(x) = 2^{nu-1} Gamma(nu) [1 - Gamma(1-nu)/Gamma(1+nu) (x/2)^{2nu} + x^2/(4(1-nu)) ...]
        const double nu = 5.0 / 6.0;
        const double t1 = std::tgamma(1.0 - nu) / std::tgamma(1.0 + nu) * std::pow(0.5 * x, 2.0 * nu);
        const double t2 = x * x / (4.0 * (1.0 - nu));
        return amp * (t1 - t2);
    }
    return amp * (1.0 - kc * std::pow(x, 5.0 / 6.0) * std::cyl_bessel_k(5.0 / 6.0, x));
}

namespace {
bool invert_small(std::vector<double> &a, int n) {   // Gauss-Jordan with partial pivoting, row-major n x n
    std::vector<double> inv((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) inv[i * n + i] = 1.0;
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r)
            if (std::fabs(a[r * n + c]) > std::fabs(a[piv * n + c])) piv = r;
        if (std::fabs(a[piv * n + c]) < 1e-300) return false;
        for (int k = 0; k < n; ++k) {
            std::swap(a[c * n + k], a[piv * n + k]);
            std::swap(inv[c * n + k], inv[piv * n + k]);
        }
        const double s = 1.0 / a[c * n + c];
        for (int k = 0; k < n; ++k) { a[c * n + k] *= s; inv[c * n + k] *= s; }
        for (int r = 0; r < n; ++r) {
            if (r == c) continue;
            const double f = a[r * n + c];
            if (f == 0.0) continue;
            for (int k = 0; k < n; ++k) { a[r * n + k] -= f * a[c * n + k]; inv[r * n + k] -= f * inv[c * n + k]; }
        }
    }
    a = inv;
    return true;
}
}  // namespace

// ------------------------------------------------------------------------------------------------ model

static double cone_gamma(double h, double h_gs) { return std::isinf(h_gs) ? 1.0 : (h_gs - h) / h_gs; }

int build_model(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, const tomo_noise *noise,
                int slope_model, int pad, int pad_os, HostModel &m, std::string &err, int layered, double fov_radius_arcsec) {
    if (!g || !cn2) { err = "geometry / cn2 is NULL"; return TOMO_EINVAL; }
    if (g->n < 2 || g->n > 512 || !(g->D > 0)) { err = "need 2 <= n <= 512 and D > 0"; return TOMO_EINVAL; }
    if (g->n_wfs < 1 || g->n_wfs > 16 || !g->wfs) { err = "need 1 <= n_wfs <= 16"; return TOMO_EINVAL; }
    if (cn2->n_layers < 1 || !cn2->h || !cn2->frac) { err = "need n_layers >= 1"; return TOMO_EINVAL; }
    if (!(r0 > 0) || !(L0 > 0)) { err = "r0 and L0 must be positive"; return TOMO_EINVAL; }
    if (g->n_targets < 0 || (g->n_targets > 0 && !g->target_xy)) { err = "bad targets"; return TOMO_EINVAL; }
    if (g->n_lo < 0 || (g->n_lo > 0 && !g->lo_wfs)) { err = "bad low-order sensor list"; return TOMO_EINVAL; }
    if (slope_model != TOMO_HUDGIN && slope_model != TOMO_FRIED && slope_model != TOMO_FFTMODEL) { err = "unknown slope model"; return TOMO_EINVAL; }
    if (g->obstruction < 0 || g->obstruction >= 1) { err = "obstruction must be in [0,1)"; return TOMO_EINVAL; }
    if (layered && g->n_targets != 0) { err = "a layered plan estimates layers, not targets: n_targets must be 0"; return TOMO_EINVAL; }
    if (layered && !(fov_radius_arcsec >= 0)) { err = "fov_radius must be >= 0"; return TOMO_EINVAL; }
    m = HostModel();
    m.n = g->n; m.D = g->D; m.d = g->D / g->n; m.r0 = r0; m.L0 = L0; m.obstruction = g->obstruction;
    m.n_wfs = g->n_wfs; m.C = 2 * g->n_wfs; m.K = cn2->n_layers; m.T = g->n_targets; m.slope_model = slope_model;
    // high-order set: all NGS or all LGS at ONE altitude, otherwise Sigma_ss is not 2RBT (L158)
    m.h_gs = g->wfs[0].h_gs;
    for (int i = 0; i < m.n_wfs; ++i) {
        const tomo_wfs &w = g->wfs[i];
        if (!(w.h_gs > 0)) { err = "guide-star altitude must be positive (INFINITY = NGS)"; return TOMO_EINVAL; }
        const bool same = (std::isinf(w.h_gs) && std::isinf(m.h_gs)) || w.h_gs == m.h_gs;
        if (!same) { err = "high-order WFSs mix NGS/LGS or LGS altitudes: not a 2RBT system (L158)"; return TOMO_EUNSUPPORTED; }
        if (w.n_remove != 0 && w.n_remove != 2 && w.n_remove != 3) { err = "n_remove must be 0, 2 or 3"; return TOMO_EINVAL; }
        m.ax.push_back(w.ax * kArcsec); m.ay.push_back(w.ay * kArcsec); m.n_remove.push_back(w.n_remove);
    }
    for (int i = 0; i < g->n_lo; ++i)   // split low-order loop sensors (L321, L412): validated, not in the CG system
        if (!std::isinf(g->lo_wfs[i].h_gs)) { err = "low-order sensors must be natural guide stars"; return TOMO_EINVAL; }
    m.lgs = !std::isinf(m.h_gs);
    double fsum = 0.0, gmin = 1.0;
    for (int k = 0; k < m.K; ++k) {
        const double hk = cn2->h[k], fk = cn2->frac[k];
        if (!(hk >= 0) || !(fk >= 0)) { err = "layer altitude / fraction negative"; return TOMO_EINVAL; }
        if (m.lgs && hk >= m.h_gs) { err = "layer at or above the guide-star altitude"; return TOMO_EINVAL; }
        m.h.push_back(hk); m.frac.push_back(fk); m.gamma.push_back(cone_gamma(hk, m.h_gs));
        gmin = std::min(gmin, m.gamma.back());
        fsum += fk;
    }
    if (std::fabs(fsum - 1.0) > 1e-9) { err = "Cn2 fractions do not sum to 1"; return TOMO_EINVAL; }
    m.layered = layered != 0;
    if (m.layered) { m.T = 1; m.bx.push_back(0.0); m.by.push_back(0.0); }   // the grid of Eq.16 with beta = 0 (reading G31)
    else for (int t = 0; t < m.T; ++t) { m.bx.push_back(g->target_xy[2 * t] * kArcsec); m.by.push_back(g->target_xy[2 * t + 1] * kArcsec); }

    // masks: subaperture valid iff its centre is inside the pupil (reading G12); phase point valid iff it is a
    // corner of a valid subaperture (Fig.2)
    const int n = m.n;
    m.smask.assign((size_t)n * n, 0);
    for (int y = 0; y < n; ++y)
        for (int x = 0; x < n; ++x) {
            bool ok;
            if (g->subap_mask) ok = g->subap_mask[y * n + x] != 0;
            else {
                const long kx = 2 * x - (n - 1), ky = 2 * y - (n - 1), r2 = kx * kx + ky * ky;
                ok = r2 <= (long)n * n;
                if (g->obstruction > 0) ok = ok && (double)r2 >= (g->obstruction * n) * (g->obstruction * n);
            }
            m.smask[y * n + x] = ok;
        }
    m.pmask.assign((size_t)(n + 1) * (n + 1), 0);
    m.row_ptr.assign(n + 1, 0);
    for (int y = 0; y < n; ++y) {
        m.row_ptr[y] = (int)m.sub_idx.size();
        for (int x = 0; x < n; ++x)
            if (m.smask[y * n + x]) {
                m.sub_idx.push_back(y * n + x); m.ix.push_back(x); m.iy.push_back(y);
                m.pmask[y * (n + 1) + x] = m.pmask[y * (n + 1) + x + 1] = 1;
                m.pmask[(y + 1) * (n + 1) + x] = m.pmask[(y + 1) * (n + 1) + x + 1] = 1;
            }
    }
    m.nv = (int)m.sub_idx.size();
    m.row_ptr[n] = m.nv;
    if (m.nv < 3) { err = "fewer than 3 valid subapertures"; return TOMO_EINVAL; }
    for (int y = 0; y <= n; ++y)
        for (int x = 0; x <= n; ++x)
            if (m.pmask[y * (n + 1) + x]) { m.ph_idx.push_back(y * (n + 1) + x); m.pix.push_back(x); m.piy.push_back(y); }
    m.nvp = (int)m.ph_idx.size();

    // n' (L179, L295; reading G19): smallest integer >= n/gamma_min + 1 with the parity of n+1
    // layered plans (L199; reading G31): the grid covers the meta-pupil D + 2 h_k theta of every layer at spacing gamma_k d
    {
        double v = n / gmin + 1.0;
        if (m.layered)
            for (int k = 0; k < m.K; ++k)
                v = std::max(v, (m.D + 2.0 * m.h[k] * fov_radius_arcsec * kArcsec) / (m.gamma[k] * m.d) + 1.0);
        int np = (int)std::ceil(v - 1e-9);
        if ((np - (n + 1)) % 2 != 0) ++np;
        m.n_p = np;
    }
    m.Kp = m.per_layer() ? m.K : 1;
    m.P = pad > 0 ? pad : next_fft_size(2 * n - 1);
    m.P_os = pad_os > 0 ? pad_os : next_fft_size(m.n_p + n - 1);
    if (m.P % 2 || !is_5smooth(m.P) || m.P_os % 2 || !is_5smooth(m.P_os)) {
        err = "FFT edge must be even and of the form 2^a 3^b 5^c"; return TOMO_EUNSUPPORTED;
    }
    if (m.P < 2 * n - 1 || m.P_os < m.n_p + n - 1) { err = "FFT edge smaller than the linear-convolution support"; return TOMO_EINVAL; }
    if (m.P > 1024 || m.P_os > 1024) { err = "FFT edge above 1024 not supported"; return TOMO_EUNSUPPORTED; }
    m.Ph = m.P / 2 + 1; m.Ph_os = m.P_os / 2 + 1; m.n_pair = m.C * (m.C + 1) / 2;

    // Eq.36 (L325): Z_{s,i} = [tip | tilt | focus] over the valid subapertures, G = (Z^T Z)^-1  (reading G14)
    double sx = 0, sy = 0, sxx = 0;
    for (int q = 0; q < m.nv; ++q) {
        const double x = (m.ix[q] - (n - 1) / 2.0) * m.d, y = (m.iy[q] - (n - 1) / 2.0) * m.d;
        sx += x; sy += y; sxx += x * x + y * y;
    }
    m.Gs.assign((size_t)m.n_wfs * 9, 0.0);
    for (int i = 0; i < m.n_wfs; ++i) {
        const int nr = m.n_remove[i];
        if (nr == 0) continue;
        const double full[9] = {(double)m.nv, 0, sx, 0, (double)m.nv, sy, sx, sy, sxx};
        std::vector<double> a((size_t)nr * nr);
        for (int r = 0; r < nr; ++r) for (int c = 0; c < nr; ++c) a[r * nr + c] = full[r * 3 + c];
        if (!invert_small(a, nr)) { err = "singular slope modal matrix"; return TOMO_EINVAL; }
        for (int r = 0; r < nr; ++r) for (int c = 0; c < nr; ++c) m.Gs[i * 9 + r * 3 + c] = a[r * nr + c];
    }
    // phase space: Z_phi = [1, x, y (, x^2+y^2)]; NGS-only systems remove piston only (reading G14)
    m.n_remove_phase = m.lgs ? *std::max_element(m.n_remove.begin(), m.n_remove.end()) : 0;
    {
        const int nc = 1 + m.n_remove_phase;
        std::vector<double> a((size_t)nc * nc, 0.0);
        for (int p = 0; p < m.nvp; ++p) {
            const double x = (m.pix[p] - n / 2.0) * m.d, y = (m.piy[p] - n / 2.0) * m.d;
            const double z[4] = {1.0, x, y, x * x + y * y};
            for (int r = 0; r < nc; ++r) for (int c = 0; c < nc; ++c) a[r * nc + c] += z[r] * z[c];
        }
        if (!invert_small(a, nc)) { err = "singular phase modal matrix"; return TOMO_EINVAL; }
        m.Gphi.assign(16, 0.0);
        for (int r = 0; r < nc; ++r) for (int c = 0; c < nc; ++c) m.Gphi[r * 4 + c] = a[r * nc + c];
    }
    // noise (L110, L260; reading G15)
    m.slope_var = model_slope_variance(m);
    m.sigma2_wfs.assign(m.n_wfs, 0.0);
    m.sigma2_full.assign((size_t)m.C * m.nv, 0.0);
    if (noise && noise->sigma2_subap) {
        for (size_t e = 0; e < m.sigma2_full.size(); ++e) {
            if (!(noise->sigma2_subap[e] >= 0)) { err = "negative noise variance"; return TOMO_EINVAL; }
            m.sigma2_full[e] = noise->sigma2_subap[e];
        }
        for (int i = 0; i < m.n_wfs; ++i) m.sigma2_wfs[i] = m.sigma2_full[(size_t)2 * i * m.nv];
        if (noise->sigma_xy_subap) {     // elongated LGS spots (L331-333): 2 x 2 block [[sxx, sxy], [sxy, syy]] per subaperture
            m.sigma_xy.assign(noise->sigma_xy_subap, noise->sigma_xy_subap + (size_t)m.n_wfs * m.nv);
            for (int i = 0; i < m.n_wfs; ++i)
                for (int e = 0; e < m.nv; ++e) {
                    const double sxx = m.sigma2_full[(size_t)2 * i * m.nv + e], syy = m.sigma2_full[(size_t)(2 * i + 1) * m.nv + e];
                    const double sxy = m.sigma_xy[(size_t)i * m.nv + e];
                    if (!(sxy * sxy <= sxx * syy * (1.0 + 1e-12))) { err = "noise block is not positive semi-definite"; return TOMO_EINVAL; }
                }
        }
    } else {
        if (noise && noise->sigma_xy_subap) { err = "sigma_xy_subap needs sigma2_subap"; return TOMO_EINVAL; }
        for (int i = 0; i < m.n_wfs; ++i) {
            double s2 = 0.0;
            if (noise && noise->sigma2_wfs) s2 = noise->sigma2_wfs[i];
            else if (noise) s2 = noise->noise_frac * m.slope_var;
            if (!(s2 >= 0)) { err = "negative noise variance"; return TOMO_EINVAL; }
            m.sigma2_wfs[i] = s2;
            for (int e = 0; e < 2 * m.nv; ++e) m.sigma2_full[(size_t)2 * i * m.nv + e] = s2;
        }
    }
    m.out_len = m.layered ? (size_t)m.Kp * m.n_p * m.n_p : (size_t)m.T * m.nvp;
    // I'_k (Eq.16; readings G18-G19): per-axis bilinear taps of the original phase points on the n' grid of
    // spacing d_k centred on the target footprint: position r_p/d_k + (n'-1)/2, independent of the target
    m.interp_i0.assign((size_t)m.Kp * (n + 1), 0);
    m.interp_w.assign((size_t)m.Kp * (n + 1), 0.0);
    for (int k = 0; k < m.Kp; ++k) {
        const double dk = (m.lgs ? m.gamma[k] : 1.0) * m.d;
        for (int a = 0; a <= n; ++a) {
            const double t = (a - n / 2.0) * m.d / dk + (m.n_p - 1) / 2.0;
            int i0 = (int)std::floor(t + 1e-12);
            i0 = std::min(std::max(i0, 0), m.n_p - 2);
            const double w = t - i0;
            if (w < -1e-9 || w > 1 + 1e-9) { err = "phase point outside the resampled grid"; return TOMO_EINVAL; }
            m.interp_i0[(size_t)k * (n + 1) + a] = i0;
            m.interp_w[(size_t)k * (n + 1) + a] = w;
        }
    }
    return TOMO_OK;
}
}  // namespace tomo
