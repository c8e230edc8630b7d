// tomo_kernels.cuh -- sm_100a kernels of the hot path (rows A1-A8 of DESIGN.md).
//
// Data flow of one Sigma_ss product (Eq.30 L267 in its zero-padded 2-D form, reading G10):
//   rows_fwd : scatter valid slopes of two image rows into one complex sequence (S_1, Eq.18-19),
//              length-P FFT along x, split into the two Hermitian half-spectra  -> T1[f][c][kx][y]
//   cols     : for one kx and ALL channels: length-P FFT along y, per-frequency C x C block product with the
//              Hermitian-packed kernel spectra (Eq.22, Eq.30), inverse FFT along y -> T2[f][c][kx][y<n]
//   rows_inv : merge two half-spectra, inverse FFT along x, crop + pupil mask (S_2, W_s; Eq.24-27, Eq.34),
//              add Sigma_eta p (L260; 2 x 2 blocks for elongated LGS spots, L331-333), reduction partials for the mode removal (Eq.36) and p.q
//   update   : alpha, x += alpha p, r -= alpha M_s q, partial r.r        (S2.G L337)
// The next rows_fwd finishes the iteration (beta, p = r + beta p) before scattering p.
// One warp owns one 1-D transform (fft_device.cuh); kernels are templated on the arithmetic type T and the
// spectrum storage type S.
#pragma once
#include <cuda_runtime.h>

#include "fft_device.cuh"

namespace tomo {

struct DevGeom {
    int n, C, N, nv, nvp, T, Kp, n_p, npairs;   // npairs = ceil(n/2) row pairs per channel image
    double d;
    const int *row_ptr;      // [n+1]
    const int *ix, *iy;      // [nv]
    const int *pix, *piy;    // [nvp]
    const int *n_remove;     // [N]
    const double *Gs;        // [N][9]   (Z_s^T Z_s)^-1
    const double *Gphi;      // [16]     (Z_phi^T Z_phi)^-1
    int n_remove_phase;
};

template <typename T> struct Stage {            // one padded FFT size: P (Sigma_ss) or P_os (Sigma_phi-s)
    FftDesc fd;
    int P, Ph;
    const typename cx_of<T>::type *tw;          // device [P], exp(-2 pi i t/P)
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// deterministic sum of `cnt` doubles by one warp (every lane returns the total)
__device__ __forceinline__ double warp_sum_array(const double *a, int cnt, int lane) {
    double s = 0.0;
    for (int i = lane; i < cnt; i += 32) s += a[i];
    return warp_sum(s);
}

template <typename T> __device__ __forceinline__ void load_twiddles(typename cx_of<T>::type *dst, const Stage<T> &st) {
    for (int i = threadIdx.x; i < st.P; i += blockDim.x) dst[i] = st.tw[i];
}

// ------------------------------------------------------------------------------------------------ rows_fwd
template <typename T> struct RowsFwdArgs {
    Stage<T> st;
    DevGeom g;
    int F;                      // frames
    T *p;                       // [F][C][nv]  search direction (read; written when update != 0)
    const T *r;                 // [F][C][nv]  residual (update only)
    typename cx_of<T>::type *T1;   // [F][C][Ph][n]
    // CG bookkeeping (update / record only)
    int update;                 // 1: beta = rho_k/rho_{k-1}, p = r + beta p before the scatter
    int record;                 // 1: rho_k = sum(partials_r) is written to hist[f][k]
    int k;                      // iteration index
    int hist_stride;            // doubles per frame in hist
    const double *partials_r;   // [F][part_stride]
    int n_part, part_stride;
    double *hist;               // [F][hist_stride]  rho_k
    const double *alpha;        // [F]  alpha of the iteration just finished; 0 marks a breakdown (freeze, G16)
};

template <typename T>
__global__ void __launch_bounds__(128) k_rows_fwd(RowsFwdArgs<T> a) {
    typedef typename cx_of<T>::type C2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, n = a.g.n, nv = a.g.nv, C = a.g.C, npairs = a.g.npairs;
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NW = blockDim.x >> 5;
    C2 *A = tw + P + (size_t)warp * 2 * P, *B = A + P;
    load_twiddles<T>(tw, a.st);
    __syncthreads();
    const int items = a.F * C * npairs;
    for (int it = blockIdx.x * NW + warp; it < items; it += gridDim.x * NW) {
        const int f = it / (C * npairs), rem = it - f * C * npairs, c = rem / npairs, j = rem - c * npairs;
        const int y0 = 2 * j, y1 = 2 * j + 1;
        T beta = (T)0;
        bool upd = false;
        if (a.record || a.update) {
            const double rho = warp_sum_array(a.partials_r + (size_t)f * a.part_stride, a.n_part, lane);
            if (a.record && rem == 0 && lane == 0) a.hist[(size_t)f * a.hist_stride + a.k] = rho;
            if (a.update) {
                const double rho_prev = a.hist[(size_t)f * a.hist_stride + a.k - 1];
                upd = (a.alpha[f] != 0.0) && rho_prev > 0.0;
                beta = upd ? (T)(rho / rho_prev) : (T)0;
            }
        }
        for (int i = lane; i < P; i += 32) A[i] = mk<T>((T)0, (T)0);
        __syncwarp();
        T *pv = a.p + ((size_t)f * C + c) * nv;
        const T *rv = a.r + ((size_t)f * C + c) * nv;
        {
            const int s0 = a.g.row_ptr[y0], e0 = a.g.row_ptr[y0 + 1];
            for (int i = s0 + lane; i < e0; i += 32) {
                T v = pv[i];
                if (upd) { v = rv[i] + beta * v; pv[i] = v; }
                A[a.g.ix[i]].x = v;
            }
        }
        if (y1 < n) {
            const int s1 = a.g.row_ptr[y1], e1 = a.g.row_ptr[y1 + 1];
            for (int i = s1 + lane; i < e1; i += 32) {
                T v = pv[i];
                if (upd) { v = rv[i] + beta * v; pv[i] = v; }
                A[a.g.ix[i]].y = v;
            }
        }
        C2 *Z = warp_fft<T, false>(A, B, a.st.fd, tw, lane);
        C2 *out = a.T1 + ((size_t)f * C + c) * Ph * n;
        for (int k = lane; k < Ph; k += 32) {
            const C2 z1 = Z[k], z2 = Z[k == 0 ? 0 : P - k];
            // row y0: (z1 + conj z2)/2 ; row y1: (z1 - conj z2)/(2i)
            out[(size_t)k * n + y0] = mk<T>((T)0.5 * (z1.x + z2.x), (T)0.5 * (z1.y - z2.y));
            if (y1 < n) out[(size_t)k * n + y1] = mk<T>((T)0.5 * (z1.y + z2.y), (T)-0.5 * (z1.x - z2.x));
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------ cols
template <typename T, typename S> struct ColsArgs {
    Stage<T> st;
    DevGeom g;
    const typename cx_of<T>::type *T1;     // [F][C][Ph][n]
    typename cx_of<T>::type *T2;           // [F][C][Ph][n]
    const typename cx_of<S>::type *spec;   // [Ph][n_pair][P], pair (co <= ci) -> co*C - co(co-1)/2 + ci - co
    int n_pair;
};

template <typename T, typename S>
__global__ void __launch_bounds__(512) k_cols(ColsArgs<T, S> a) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, n = a.g.n, C = a.g.C;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NW = blockDim.x >> 5;
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    C2 *X = tw + P, *Y = X + (size_t)C * P, *scr = Y + (size_t)C * P + (size_t)warp * P;
    const int kx = blockIdx.x, f = blockIdx.y;
    load_twiddles<T>(tw, a.st);
    __syncthreads();
    const bool even = (a.st.fd.nrad & 1) == 0;
    for (int c = warp; c < C; c += NW) {       // forward along y, result lands in X[c]
        C2 *dst = X + (size_t)c * P;
        C2 *in = even ? dst : scr, *other = even ? scr : dst;
        const C2 *src = a.T1 + (((size_t)f * C + c) * Ph + kx) * n;
        for (int i = lane; i < P; i += 32) in[i] = (i < n) ? src[i] : mk<T>((T)0, (T)0);
        warp_fft<T, false>(in, other, a.st.fd, tw, lane);
    }
    __syncthreads();
    // y~_co(f) = sum_ci theta~_{co,ci}(f) p~_ci(f)   (Eq.30); theta~_{ci,co} = conj(theta~_{co,ci})
    const S2 *Sk = a.spec + (size_t)kx * a.n_pair * P;
    for (int o = threadIdx.x; o < C * P; o += blockDim.x) {
        const int co = o / P, ky = o - co * P;
        T ar = (T)0, ai = (T)0;
        for (int ci = 0; ci < C; ++ci) {
            const int lo = ci < co ? ci : co, hi = ci < co ? co : ci;
            const S2 s = Sk[(size_t)(lo * C - (lo * (lo - 1)) / 2 + (hi - lo)) * P + ky];
            const C2 xv = X[(size_t)ci * P + ky];
            const T sr = (T)s.x, si = (ci < co) ? -(T)s.y : (T)s.y;
            ar += sr * xv.x - si * xv.y;
            ai += sr * xv.y + si * xv.x;
        }
        Y[o] = mk<T>(ar, ai);
    }
    __syncthreads();
    for (int c = warp; c < C; c += NW) {       // inverse along y, keep rows y < n
        C2 *res = warp_fft<T, true>(Y + (size_t)c * P, scr, a.st.fd, tw, lane);
        C2 *dst = a.T2 + (((size_t)f * C + c) * Ph + kx) * n;
        for (int i = lane; i < n; i += 32) dst[i] = res[i];
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------ rows_inv
#define TOMO_NRED 5     // per (channel, row pair): p.q, sum q, sum p, sum coord*q, sum coord*p

template <typename T> struct RowsInvArgs {
    Stage<T> st;
    DevGeom g;
    int F;
    const typename cx_of<T>::type *T2;   // [F][C][Ph][n]
    const T *p;                          // [F][C][nv]
    const T *sigma2;                     // [C][nv]  diagonal of Sigma_eta
    const T *sigma_xy;                   // [N][nv]  x-y noise covariance per subaperture (elongated LGS spots, L331-333) or NULL
    T *q;                                // [F][C][nv]  W (Sigma_ss + Sigma_eta) W^T p, modes not yet removed
    double *partials_q;                  // [F][C][npairs][TOMO_NRED]
};

template <typename T>
__global__ void __launch_bounds__(128) k_rows_inv(RowsInvArgs<T> a) {
    typedef typename cx_of<T>::type C2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, n = a.g.n, nv = a.g.nv, C = a.g.C, npairs = a.g.npairs;
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NW = blockDim.x >> 5;
    C2 *A = tw + P + (size_t)warp * 2 * P, *B = A + P;
    load_twiddles<T>(tw, a.st);
    __syncthreads();
    const int items = a.F * C * npairs;
    const T half_n = (T)(0.5 * (n - 1));
    for (int it = blockIdx.x * NW + warp; it < items; it += gridDim.x * NW) {
        const int f = it / (C * npairs), rem = it - f * C * npairs, c = rem / npairs, j = rem - c * npairs;
        const int y0 = 2 * j, y1 = 2 * j + 1;
        const bool two = y1 < n;
        const C2 *src = a.T2 + ((size_t)f * C + c) * Ph * n;
        for (int k = lane; k < Ph; k += 32) {
            const C2 u = src[(size_t)k * n + y0];
            const C2 v = two ? src[(size_t)k * n + y1] : mk<T>((T)0, (T)0);
            A[k] = mk<T>(u.x - v.y, u.y + v.x);                            // U_k + i V_k
            if (k > 0 && 2 * k < P) A[P - k] = mk<T>(u.x + v.y, v.x - u.y);   // conj(U_k) + i conj(V_k)
        }
        C2 *Z = warp_fft<T, true>(A, B, a.st.fd, tw, lane);
        const size_t base = ((size_t)f * C + c) * nv;
        const int comp = c & 1;
        double s_pq = 0, s_q = 0, s_p = 0, s_fq = 0, s_fp = 0;
        for (int row = 0; row < (two ? 2 : 1); ++row) {
            const int y = row ? y1 : y0;
            const int s0 = a.g.row_ptr[y], e0 = a.g.row_ptr[y + 1];
            for (int i = s0 + lane; i < e0; i += 32) {
                const int x = a.g.ix[i];
                const T pv = a.p[base + i];
                T qv = (row ? Z[x].y : Z[x].x) + a.sigma2[(size_t)c * nv + i] * pv;
                if (a.sigma_xy)          // 2 x 2 noise block: the other slope component of the same subaperture
                    qv += a.sigma_xy[(size_t)(c >> 1) * nv + i] * a.p[((size_t)f * C + (c ^ 1)) * nv + i];
                a.q[base + i] = qv;
                const T coord = ((comp ? (T)y : (T)x) - half_n) * (T)a.g.d;
                s_pq += (double)pv * (double)qv; s_q += (double)qv; s_p += (double)pv;
                s_fq += (double)coord * (double)qv; s_fp += (double)coord * (double)pv;
            }
        }
        s_pq = warp_sum(s_pq); s_q = warp_sum(s_q); s_p = warp_sum(s_p); s_fq = warp_sum(s_fq); s_fp = warp_sum(s_fp);
        if (lane == 0) {
            double *o = a.partials_q + (size_t)it * TOMO_NRED;
            o[0] = s_pq; o[1] = s_q; o[2] = s_p; o[3] = s_fq; o[4] = s_fp;
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------ update
template <typename T> struct UpdateArgs {
    DevGeom g;
    T *x, *r;                  // [F][C][nv]
    const T *p, *q;
    const double *partials_q;  // [F][C][npairs][TOMO_NRED]
    const double *hist;        // rho_k at hist[f*hist_stride + k]
    int hist_stride, k;
    double *alpha;             // [F]
    double *partials_r;        // [F][part_stride], gridDim.x entries written
    int part_stride;
};

// per-WFS mode coefficients a = G Z^T q and the projected p.q from the rows_inv partials (Eq.36):
// M q = q - Z a; p.(M q) = p.q - (Z^T p)^T G (Z^T q).  red: [C][TOMO_NRED] channel totals.
__device__ __forceinline__ double mode_coeffs(const DevGeom &g, const double *red, double *coef /*[N][3]*/) {
    double pq = 0.0;
    for (int i = 0; i < g.N; ++i) {
        const double *rx = red + (2 * i) * TOMO_NRED, *ry = red + (2 * i + 1) * TOMO_NRED;
        pq += rx[0] + ry[0];
        const double tq[3] = {rx[1], ry[1], rx[3] + ry[3]}, tp[3] = {rx[2], ry[2], rx[4] + ry[4]};
        const int nr = g.n_remove[i];
        const double *G = g.Gs + i * 9;
        for (int u = 0; u < 3; ++u) {
            double s = 0.0;
            if (u < nr) for (int v = 0; v < nr; ++v) s += G[u * 3 + v] * tq[v];
            coef[i * 3 + u] = s;
            if (u < nr) pq -= tp[u] * s;
        }
    }
    return pq;
}

template <typename T>
__global__ void __launch_bounds__(256) k_update(UpdateArgs<T> a) {
    __shared__ double red[32 * TOMO_NRED];
    __shared__ double coef[16 * 3];
    __shared__ double s_alpha;
    __shared__ double wsum[8];
    const int f = blockIdx.y, C = a.g.C, nv = a.g.nv, npairs = a.g.npairs;
    if (threadIdx.x < C * TOMO_NRED) {
        const int c = threadIdx.x / TOMO_NRED, v = threadIdx.x - c * TOMO_NRED;
        const double *src = a.partials_q + ((size_t)f * C + c) * npairs * TOMO_NRED + v;
        double s = 0.0;
        for (int j = 0; j < npairs; ++j) s += src[(size_t)j * TOMO_NRED];
        red[threadIdx.x] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double pq = mode_coeffs(a.g, red, coef);
        const double rho = a.hist[(size_t)f * a.hist_stride + a.k];
        const double al = (rho > 0.0 && pq > 0.0) ? rho / pq : 0.0;     // breakdown: freeze (reading G16)
        s_alpha = al;
        if (blockIdx.x == 0) a.alpha[f] = al;
    }
    __syncthreads();
    const T alpha = (T)s_alpha;
    const T half_n = (T)(0.5 * (a.g.n - 1));
    double rr = 0.0;
    const size_t base = (size_t)f * C * nv;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < C * nv; e += gridDim.x * blockDim.x) {
        const int c = e / nv, i = e - c * nv, w = c >> 1, comp = c & 1;
        const T coord = ((comp ? (T)a.g.iy[i] : (T)a.g.ix[i]) - half_n) * (T)a.g.d;
        const T qp = a.q[base + e] - ((T)coef[w * 3 + comp] + (T)coef[w * 3 + 2] * coord);
        T rv = a.r[base + e];
        if (s_alpha != 0.0) {
            a.x[base + e] += alpha * a.p[base + e];
            rv -= alpha * qp;
            a.r[base + e] = rv;
        }
        rr += (double)rv * (double)rv;
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

// rho_{n_iter} of the last iteration -> hist
static __global__ void k_finalize(const double *partials_r, int n_part, int part_stride, double *hist, int hist_stride, int k) {
    const int f = blockIdx.x, lane = threadIdx.x;
    const double rho = warp_sum_array(partials_r + (size_t)f * part_stride, n_part, lane);
    if (lane == 0) hist[(size_t)f * hist_stride + k] = rho;
}

// p = r + beta p after a single teacher-forced step (tomo_cg_step); scal = {rho_{k+1}, alpha, beta}
template <typename T>
__global__ void k_step_finish(DevGeom g, const T *r, T *p, const double *partials_r, int n_part, const double *hist,
                              const double *alpha, double *scal) {
    __shared__ double s_beta;
    if (threadIdx.x < 32) {
        const double rho1 = warp_sum_array(partials_r, n_part, threadIdx.x);
        if (threadIdx.x == 0) {
            const double rho0 = hist[0], al = alpha[0];
            const double beta = (al != 0.0 && rho0 > 0.0) ? rho1 / rho0 : 0.0;
            s_beta = beta;
            if (blockIdx.x == 0) { scal[0] = rho1; scal[1] = al; scal[2] = beta; }
        }
    }
    __syncthreads();
    if (alpha[0] == 0.0) return;
    const T beta = (T)s_beta;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < g.C * g.nv; e += gridDim.x * blockDim.x)
        p[e] = r[e] + beta * p[e];
}

}  // namespace tomo
