// tomo_kernels_minres.cuh -- MINRES recurrences (Paige & Saunders) around the same Sigma_ss product kernels.
//
// The paper keeps MINRES for the Toeplitz method (PAPER.md S2.G L337; L426 "MINRES and CG are used for the Toeplitz and
// sparse methods"; Fig.13: CG does not converge in its noise-free case).  One iteration k = 1, 2, ...:
//     q = A v_k                                  rows_fwd / cols / rows_inv on d_p = v_k   (the CG product kernels)
//     alpha_k = v_k . M_s q                      from the rows_inv partials                 (k_minres_lanczos)
//     u = M_s q - alpha_k v_k - beta_k v_{k-1}   -> d_r, partial |u|^2
//     beta_{k+1} = |u|; Givens rotation k of the Lanczos tridiagonal: delta_k, gbar_k, eps_{k+1}, dbar_{k+1}, gamma_k,
//     c_k, s_k, phi_k, phibar_k                  fp64, every CTA redundantly, fixed order    (k_minres_update)
//     w_k = (v_k - eps_k w_{k-2} - delta_k w_{k-1}) / gamma_k;  x += phi_k w_k;  v_{k-1} = v_k;  v_{k+1} = u / beta_{k+1}
// History: phibar_k^2 (= |b - A x_k|^2) at hist[k], k = 0..n_iter, so that tomo_get_residuals returns phibar_k.
// A breakdown (beta_{k+1} = 0 or gamma_k = 0) freezes the iterate, as for CG (reading G16).
//
// A is singular on span(Z) when modes are removed (G14).  In exact arithmetic every v_k lies in range(M_s); in fp32 the
// three-term recurrence lets a null-space component of v_k grow (nothing damps it: A annihilates it), and MINRES, unlike
// CG, feeds it back into x through the w_k (measured: wavefront error 3e-3 and growing with the count on a system with
// one tip/tilt-removed and one unprojected WFS; 1e-5 with the fix).  So every v_k is re-projected once, v_k <- M_s v_k,
// with the coefficients (Z^T Z)^-1 Z^T v_k that the product's reduction partials carry anyway -- a no-op in exact
// arithmetic, hence absent from the oracle.
#pragma once
#include <cuda_runtime.h>

#include "tomo_kernels.cuh"

namespace tomo {

// per-frame scalar state, double-buffered by iteration parity: written by CTA 0 of k_minres_update, read by the next
// iteration's kernels
enum { MS_BETA = 0, MS_C = 1, MS_S = 2, MS_DBAR = 3, MS_EPS = 4, MS_PHIBAR = 5, MS_FROZEN = 6, MS_N = 8 };

template <typename T> struct MinresArgs {
    DevGeom g;
    T *x, *v, *v_old, *u, *w1, *w2;     // [F][C][nv]: iterate, v_k (= the plan's d_p), v_{k-1}, u (= d_r), w_{k-1}, w_{k-2}
    const T *q;                          // [F][C][nv] W (Sigma_ss + Sigma_eta) W^T v_k, modes not yet removed
    const double *partials_q;            // [F][C][npairs][TOMO_NRED]
    double *partials_r;                  // [F][part_stride]
    int n_part, part_stride;
    double *state;                       // [2][F][MS_N]
    double *alpha;                       // [F]
    double *hist;                        // [F][hist_stride]
    int hist_stride, k, F;               // k = 0-based iteration index (the text's k - 1)
};

// v_1 = r0 / beta_1 with r0 in a.u (cold: b; warm: b - A x0), v_0 = w_0 = w_{-1} = 0, rotation state of "iteration 0"
template <typename T>
__global__ void __launch_bounds__(256) k_minres_init(MinresArgs<T> a) {
    __shared__ double s_beta;
    const int f = blockIdx.y;
    if (threadIdx.x < 32) {
        const double rr = warp_sum_array(a.partials_r + (size_t)f * a.part_stride, a.n_part, threadIdx.x);
        if (threadIdx.x == 0) {
            const double beta = sqrt(rr);
            s_beta = beta;
            if (blockIdx.x == 0) {
                double *st = a.state + (size_t)f * MS_N;          // buffer 0 is read by iteration k = 0
                st[MS_BETA] = beta; st[MS_C] = -1.0; st[MS_S] = 0.0; st[MS_DBAR] = 0.0; st[MS_EPS] = 0.0;
                st[MS_PHIBAR] = beta; st[MS_FROZEN] = beta > 0.0 ? 0.0 : 1.0;
                a.hist[(size_t)f * a.hist_stride] = rr;
            }
        }
    }
    __syncthreads();
    const double beta = s_beta;
    const T inv = beta > 0.0 ? (T)(1.0 / beta) : (T)0;
    const size_t base = (size_t)f * a.g.C * a.g.nv;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < a.g.C * a.g.nv; e += gridDim.x * blockDim.x) {
        a.v[base + e] = a.u[base + e] * inv;
        a.v_old[base + e] = (T)0; a.w1[base + e] = (T)0; a.w2[base + e] = (T)0;
    }
}

// per-WFS coefficients of BOTH q and v on the removed modes, and v . M_s q (cf. mode_coeffs)
__device__ __forceinline__ double mode_coeffs_qv(const DevGeom &g, const double *red, double *coef_q, double *coef_v) {
    double pq = 0.0;
    for (int i = 0; i < g.N; ++i) {
        const double *rx = red + (2 * i) * TOMO_NRED, *ry = red + (2 * i + 1) * TOMO_NRED;
        pq += rx[0] + ry[0];
        const double tq[3] = {rx[1], ry[1], rx[3] + ry[3]}, tp[3] = {rx[2], ry[2], rx[4] + ry[4]};
        const int nr = g.n_remove[i];
        const double *G = g.Gs + i * 9;
        for (int u = 0; u < 3; ++u) {
            double sq = 0.0, sv = 0.0;
            if (u < nr) for (int v = 0; v < nr; ++v) { sq += G[u * 3 + v] * tq[v]; sv += G[u * 3 + v] * tp[v]; }
            coef_q[i * 3 + u] = sq; coef_v[i * 3 + u] = sv;
            if (u < nr) pq -= tp[u] * sq;
        }
    }
    return pq;
}

// alpha_k and the unnormalised next Lanczos vector u (mode removal Eq.36 L325 folded in, as in k_update); v_k <- M_s v_k
template <typename T>
__global__ void __launch_bounds__(256) k_minres_lanczos(MinresArgs<T> a) {
    __shared__ double red[32 * TOMO_NRED];
    __shared__ double coef[16 * 3], coefv[16 * 3];
    __shared__ double s_alpha;
    __shared__ double wsum[8];
    const int f = blockIdx.y, C = a.g.C, nv = a.g.nv, npairs = a.g.npairs;
    const double *st = a.state + ((size_t)(a.k & 1) * a.F + f) * MS_N;
    if (threadIdx.x < C * TOMO_NRED) {
        const int c = threadIdx.x / TOMO_NRED, v = threadIdx.x - c * TOMO_NRED;
        const double *src = a.partials_q + ((size_t)f * C + c) * npairs * TOMO_NRED + v;
        double s = 0.0;
        for (int j = 0; j < npairs; ++j) s += src[(size_t)j * TOMO_NRED];
        red[threadIdx.x] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double vq = mode_coeffs_qv(a.g, red, coef, coefv);          // v . M_s q
        s_alpha = vq;
        if (blockIdx.x == 0) a.alpha[f] = vq;
    }
    __syncthreads();
    const bool frozen = st[MS_FROZEN] != 0.0;
    const T alpha = (T)s_alpha, beta = (T)st[MS_BETA];
    const T half_n = (T)(0.5 * (a.g.n - 1));
    double rr = 0.0;
    const size_t base = (size_t)f * C * nv;
    if (!frozen)
        for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < C * nv; e += gridDim.x * blockDim.x) {
            const int c = e / nv, i = e - c * nv, w = c >> 1, comp = c & 1;
            const T coord = ((comp ? (T)a.g.iy[i] : (T)a.g.ix[i]) - half_n) * (T)a.g.d;
            const T qp = a.q[base + e] - ((T)coef[w * 3 + comp] + (T)coef[w * 3 + 2] * coord);
            const T vp = a.v[base + e] - ((T)coefv[w * 3 + comp] + (T)coefv[w * 3 + 2] * coord);   // M_s v_k
            const T uv = qp - alpha * vp - beta * a.v_old[base + e];
            a.v[base + e] = vp;
            a.u[base + e] = uv;
            rr += (double)uv * (double)uv;
        }
    rr = warp_sum(rr);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = rr;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += wsum[w];
        a.partials_r[(size_t)f * a.part_stride + blockIdx.x] = s;
    }
}

// rotation k, w_k, x_k, and the shift of the Lanczos vectors
template <typename T>
__global__ void __launch_bounds__(256) k_minres_update(MinresArgs<T> a) {
    __shared__ double sc[8];
    const int f = blockIdx.y;
    const double *st = a.state + ((size_t)(a.k & 1) * a.F + f) * MS_N;
    double *nx = a.state + ((size_t)((a.k + 1) & 1) * a.F + f) * MS_N;
    if (threadIdx.x < 32) {
        const double uu = warp_sum_array(a.partials_r + (size_t)f * a.part_stride, a.n_part, threadIdx.x);
        if (threadIdx.x == 0) {
            const double alpha = a.alpha[f], c = st[MS_C], s = st[MS_S], dbar = st[MS_DBAR], phibar = st[MS_PHIBAR];
            bool frozen = st[MS_FROZEN] != 0.0;
            const double beta_next = sqrt(uu);
            const double delta = c * dbar + s * alpha;
            const double gbar = s * dbar - c * alpha;
            const double gamma = sqrt(gbar * gbar + beta_next * beta_next);
            if (!(gamma > 0.0)) frozen = true;
            double c_new = c, s_new = s, phi = 0.0, phibar_new = phibar, eps_next = st[MS_EPS], dbar_next = dbar;
            if (!frozen) {
                c_new = gbar / gamma; s_new = beta_next / gamma;
                phi = c_new * phibar; phibar_new = s_new * phibar;
                eps_next = s * beta_next; dbar_next = -c * beta_next;
            }
            sc[0] = frozen ? 1.0 : 0.0; sc[1] = st[MS_EPS]; sc[2] = delta; sc[3] = frozen ? 0.0 : 1.0 / gamma; sc[4] = phi;
            sc[5] = (!frozen && beta_next > 0.0) ? 1.0 / beta_next : 0.0;
            if (blockIdx.x == 0) {
                nx[MS_BETA] = frozen ? st[MS_BETA] : beta_next; nx[MS_C] = c_new; nx[MS_S] = s_new; nx[MS_DBAR] = dbar_next;
                nx[MS_EPS] = eps_next; nx[MS_PHIBAR] = phibar_new;
                nx[MS_FROZEN] = (frozen || !(beta_next > 0.0)) ? 1.0 : 0.0;
                a.hist[(size_t)f * a.hist_stride + a.k + 1] = phibar_new * phibar_new;
            }
        }
    }
    __syncthreads();
    if (sc[0] != 0.0) return;
    const T eps = (T)sc[1], delta = (T)sc[2], inv_gamma = (T)sc[3], phi = (T)sc[4], inv_beta = (T)sc[5];
    const bool shift = sc[5] != 0.0;
    const size_t base = (size_t)f * a.g.C * a.g.nv;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < a.g.C * a.g.nv; e += gridDim.x * blockDim.x) {
        const T vv = a.v[base + e], w1 = a.w1[base + e], w2 = a.w2[base + e];
        const T w = (vv - eps * w2 - delta * w1) * inv_gamma;
        a.x[base + e] += phi * w;
        a.w2[base + e] = w1; a.w1[base + e] = w;
        if (shift) { a.v_old[base + e] = vv; a.v[base + e] = a.u[base + e] * inv_beta; }
    }
}

}  // namespace tomo
