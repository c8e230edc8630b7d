// lo_path.cu -- split low-order path for the NGS tip/tilt sensors (Table 2).
// The paper gives no algorithm; reading G30 of DESIGN.md: MMSE tip/tilt of each target from the aperture-mean slopes of the
// low-order sensors, R_lo built once on the host (host_kernels.cpp: build_lo_estimator), applied per frame by k_lo_addback,
// which adds tau_x x_p + tau_y y_p to the tip/tilt-free high-order wavefront (Eq.35).  Shares nothing with oracle/.
#include <cuda_runtime.h>

#include <cmath>
#include <cstring>
#include <string>
#include <vector>

#include "host_model.hpp"
#include "tomo.h"
#include "tomo_host.h"

namespace tomo {
void set_error(const std::string &s);
}
using namespace tomo;

struct tomo_lo {
    int n_lo = 0, T = 0, nvp = 0;
    float *d_R = nullptr;      // [2T][2 n_lo]
    float *d_xy = nullptr;     // [2][n_vphi] coordinates of the valid phase points [m]
};

namespace {
int lo_build(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, int slope_model, double sigma2_lo,
             HostModel &m, std::vector<double> &R, std::vector<double> &Cm) {
    if (!g || !cn2) { set_error("geometry / cn2 is NULL"); return TOMO_EINVAL; }
    if (slope_model != TOMO_HUDGIN && slope_model != TOMO_FRIED) {
        set_error("low-order estimator: stencil slope models only (TOMO_HUDGIN, TOMO_FRIED)");
        return TOMO_EUNSUPPORTED;
    }
    if (!(sigma2_lo >= 0.0)) { set_error("sigma2_lo must be >= 0"); return TOMO_EINVAL; }
    std::string err;
    tomo_noise nz;
    std::memset(&nz, 0, sizeof(nz));
    int rc = build_model(g, cn2, r0, L0, &nz, slope_model, 0, 0, m, err);
    if (rc) { set_error(err); return rc; }
    if (g->n_lo < 1) { set_error("no low-order sensor in the geometry (n_lo == 0)"); return TOMO_EINVAL; }
    if (m.T < 1) { set_error("no target direction"); return TOMO_EINVAL; }
    std::vector<double> ux, uy;
    for (int i = 0; i < g->n_lo; ++i) { ux.push_back(g->lo_wfs[i].ax * kArcsec); uy.push_back(g->lo_wfs[i].ay * kArcsec); }
    for (int t = 0; t < m.T; ++t) { ux.push_back(m.bx[t]); uy.push_back(m.by[t]); }
    rc = build_lo_estimator(m, ux, uy, g->n_lo, sigma2_lo, R, Cm);
    if (rc) set_error("C_gg + sigma2_lo I is not positive definite (coincident noiseless sensors?)");
    return rc;
}

// One thread per (valid phase point, target, frame).  tau = R_lo[2t..2t+1][:] . g is recomputed by every thread (2 x 2 n_lo
// FMAs on values that sit in L1): cheaper than a second launch.  HBM traffic: 8 B per point (read + write) + 8 B coordinates.
__global__ void k_lo_addback(const float *__restrict__ R, const float *__restrict__ xy, const float *__restrict__ g,
                             float *__restrict__ w, int n_lo, int T, int nvp) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x, t = blockIdx.y, f = blockIdx.z;
    if (p >= nvp) return;
    const int n_g = 2 * n_lo;
    const float *gf = g + (size_t)f * n_g, *Rx = R + (size_t)(2 * t) * n_g, *Ry = Rx + n_g;
    float tx = 0.f, ty = 0.f;
    for (int q = 0; q < n_g; ++q) {
        const float v = __ldg(gf + q);
        tx = fmaf(__ldg(Rx + q), v, tx);
        ty = fmaf(__ldg(Ry + q), v, ty);
    }
    const size_t o = ((size_t)f * T + t) * nvp + p;
    w[o] = fmaf(tx, __ldg(xy + p), fmaf(ty, __ldg(xy + nvp + p), w[o]));
}
}  // namespace

extern "C" int tomo_host_lo_estimator(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                                      double sigma2_lo, double *R_out, double *cov_out) {
    HostModel m;
    std::vector<double> R, Cm;
    int rc = lo_build(g, cn2, r0, L0, slope_model, sigma2_lo, m, R, Cm);
    if (rc) return rc;
    if (R_out) std::memcpy(R_out, R.data(), R.size() * sizeof(double));
    if (cov_out) std::memcpy(cov_out, Cm.data(), Cm.size() * sizeof(double));
    return TOMO_OK;
}

extern "C" int tomo_lo_create(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                              double sigma2_lo, tomo_lo **out) {
    if (!out) { set_error("out is NULL"); return TOMO_EINVAL; }
    *out = nullptr;
    HostModel m;
    std::vector<double> R, Cm;
    int rc = lo_build(g, cn2, r0, L0, slope_model, sigma2_lo, m, R, Cm);
    if (rc) return rc;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        set_error("no CUDA device: libtomo_b200 has no CPU fallback");
        return TOMO_ECUDA;
    }
    tomo_lo *lo = new tomo_lo;
    lo->n_lo = g->n_lo; lo->T = m.T; lo->nvp = m.nvp;
    std::vector<float> Rf(R.begin(), R.end()), xy((size_t)2 * m.nvp);
    for (int p = 0; p < m.nvp; ++p) {
        xy[p] = (float)((m.pix[p] - m.n / 2.0) * m.d);
        xy[(size_t)m.nvp + p] = (float)((m.piy[p] - m.n / 2.0) * m.d);
    }
    cudaError_t e = cudaMalloc(&lo->d_R, Rf.size() * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&lo->d_xy, xy.size() * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpy(lo->d_R, Rf.data(), Rf.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(lo->d_xy, xy.data(), xy.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        set_error(std::string("tomo_lo_create: ") + cudaGetErrorString(e));
        tomo_lo_destroy(lo);
        return e == cudaErrorMemoryAllocation ? TOMO_ENOMEM : TOMO_ECUDA;
    }
    *out = lo;
    return TOMO_OK;
}

extern "C" int tomo_lo_apply(const tomo_lo *lo, const float *lo_slopes, float *wavefront, int n_frames, void *cuda_stream) {
    if (!lo) { set_error("lo is NULL"); return TOMO_EINVAL; }
    if (n_frames < 0 || n_frames > 65535) { set_error("n_frames out of range [0, 65535]"); return TOMO_EINVAL; }
    if (n_frames == 0) return TOMO_OK;      // nothing to do; empty buffers may be NULL
    if (!lo_slopes || !wavefront) { set_error("NULL argument"); return TOMO_EINVAL; }
    const dim3 grid((lo->nvp + 255) / 256, lo->T, n_frames);
    k_lo_addback<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(lo->d_R, lo->d_xy, lo_slopes, wavefront, lo->n_lo, lo->T, lo->nvp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("k_lo_addback: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
    return TOMO_OK;
}

extern "C" void tomo_lo_destroy(tomo_lo *lo) {
    if (!lo) return;
    cudaFree(lo->d_R);
    cudaFree(lo->d_xy);
    delete lo;
}
