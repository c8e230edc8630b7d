// host_model.hpp -- host-side (fp64, one-time) part of libtomo_b200: problem validation, pupil masks, modal
// matrices, von Karman slope covariances, 2RBT generators and their spectra (row A0 of DESIGN.md).
// Citations are PAPER.md L<line> of arXiv:1806.07938.  Nothing here runs per frame.
#pragma once
#include <complex>
#include <cstdint>
#include <string>
#include <vector>

#include "tomo.h"

namespace tomo {

constexpr double kArcsec = 3.14159265358979323846 / (180.0 * 3600.0);

struct HostModel {
    // problem statement (S2 L41-58)
    int n = 0, n_wfs = 0, C = 0, K = 0, T = 0;
    double D = 0, d = 0, r0 = 0, L0 = 0, h_gs = 0, obstruction = 0;
    bool lgs = false;
    bool layered = false;                // layered-phase (MCAO) plan (L199; reading G31): T = 1 pseudo-target on the axis,
                                         // layers kept apart, n_p = n_m, no I'_k / W_phi / M_phi
    bool per_layer() const { return lgs || layered; }
    int slope_model = TOMO_HUDGIN;
    std::vector<double> ax, ay;          // WFS directions [rad]
    std::vector<double> bx, by;          // target directions [rad]
    std::vector<int> n_remove;           // per WFS
    std::vector<double> h, frac, gamma;  // layers; gamma_k = (h_gs - h_k)/h_gs (L158)
    // masks (Fig.2)
    std::vector<uint8_t> smask, pmask;   // n*n, (n+1)*(n+1)
    std::vector<int> sub_idx, ph_idx;    // row-major grid index of valid entries
    std::vector<int> ix, iy;             // grid coordinates of valid subapertures
    std::vector<int> row_ptr;            // [n+1] first valid entry of each subaperture row
    std::vector<int> pix, piy;           // grid coordinates of valid phase points
    int nv = 0, nvp = 0;
    // FFT sizes
    int n_p = 0;                         // n' (L179, L295; reading G19)
    int Kp = 0;                          // layers kept apart in the phi-s product: K (LGS, layered) or 1 (NGS)
    size_t out_len = 0;                  // fp32 values one frame's projection writes: T * nvp, layered: K * n_p * n_p
    int P = 0, Ph = 0, P_os = 0, Ph_os = 0, n_pair = 0;
    // mode removal (Eq.36): per WFS G = (Z^T Z)^-1, row-major 3x3 (unused rows/cols zero)
    std::vector<double> Gs;              // [n_wfs][9]
    int n_remove_phase = 0;              // columns of Z_phi beyond piston: 0, 2 or 3
    std::vector<double> Gphi;            // [16] (Z_phi^T Z_phi)^-1 padded to 4x4
    // noise (L110, L260)
    std::vector<double> sigma2_wfs;      // [n_wfs]
    std::vector<double> sigma2_full;     // [C][nv]
    std::vector<double> sigma_xy;        // [n_wfs][nv] x-y noise covariance per subaperture (L331-333), empty = diagonal noise
    double slope_var = 0;                // 1/2 [theta_x0x0(0) + theta_y0y0(0)]
    // bilinear tables I'_k, separable per axis (Eq.16; reading G18): [Kp][n+1]
    std::vector<int> interp_i0;
    std::vector<double> interp_w;
};

// Fill a HostModel from the ABI structs; returns TOMO_OK or an error code and sets `err`.
int build_model(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, const tomo_noise *noise,
                int slope_model, int pad, int pad_os, HostModel &m, std::string &err, int layered = 0,
                double fov_radius_arcsec = 0.0);

// D_phi(r) of Eq.53 (L619) with the exact prefactor (reading G2).
double structure_function(double r, double r0, double L0);

// theta[(i,a),(j,b)](l): fills gen[C][C][L][L] (L = 2n-1); only blocks with channel(i,a) <= channel(j,b) are
// computed, the lower blocks are filled by theta_{ba}(l) = theta_{ab}(-l).
void build_css_generators(const HostModel &m, std::vector<double> &gen);

// xi'[k,(j,b)](l) for one target: gen[Kp][C][Los][Los], Los = n'+n-1.
void build_cos_generators(const HostModel &m, int target, std::vector<double> &gen);

// Low-order NGS tip/tilt estimator (reading G30; L321, L412): directions (ux, uy) [rad] = n_lo sensors then the T targets.
// Cm: covariance of the aperture-mean slope pairs [2M][2M]; R = C_tau,g (C_gg + sigma2_lo I)^-1, [2T][2 n_lo] row-major.
// Returns TOMO_EINVAL when C_gg + sigma2_lo I is not positive definite.
int build_lo_estimator(const HostModel &m, const std::vector<double> &ux, const std::vector<double> &uy, int n_lo,
                       double sigma2_lo, std::vector<double> &R, std::vector<double> &Cm);

// 1/2 [theta_x0x0(0) + theta_y0y0(0)] without building the whole table.
double model_slope_variance(const HostModel &m);

// Spectrum of one generator: circular embedding K[(-l) mod P] = g(l) (reading G10), 2-D real DFT in fp64, times
// 1/P^2 (G24), Hermitian half in x.  g: [Lo+Li-1][Lo+Li-1] with index (ly + Lo-1, lx + Lo-1), l in [-(Lo-1), Li-1]^2.
// out[kx][ky], kx in [0, P/2], ky in [0, P).
void generator_spectrum(const double *g, int n_out, int n_in, int P, std::complex<double> *out);

// in-place fp64 complex FFT of 5-smooth length (forward: exp(-2 pi i jk/n)).
void host_fft(std::complex<double> *x, int n, int stride, bool inverse);

bool is_5smooth(int v);
int next_fft_size(int v);                // smallest even 5-smooth integer >= v

}  // namespace tomo
