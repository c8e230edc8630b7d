// tomo_kernels_cos.cuh -- projectors (A1, A5 stand-alone, A8) and the target projection Sigma_phi-s zeta (A7).
//
// A7 follows PAPER.md Eq.32 (L290) / Eq.31 (L276): zeta~_c = F[S_1 zeta_c] once at P_os (rows_fwd + cos_cols_fwd);
// per target t and layer k:  g~ = sum_c xi~'_{t,k,c} . zeta~_c  (cos_mac_inv: spectra streamed from HBM once,
// inverse FFT along y), inverse FFT along x cropped to the n' x n' grid (cos_rows_inv), then the 4-tap bilinear
// I'_k gather summed over layers (cos_gather).  NGS systems run the same kernels with one summed "layer".
#pragma once
#include "tomo_kernels.cuh"

namespace tomo {

// ------------------------------------------------------------------------------------------------ M_s v
// out = M_s v = v - Z (Z^T Z)^-1 Z^T v per WFS (Eq.36; tip = 1 on x-slopes, tilt = 1 on y-slopes,
// focus = (x_q, y_q); reading G14).  One CTA per (wfs, frame).  Optionally also writes copies (r, p of the CG
// start), zeroes x, and leaves sum(out^2) of the WFS in partials_r[f][wfs] (rho_0 = b.b).
template <typename Tin, typename Tout> struct ProjectArgs {
    DevGeom g;
    const Tin *in;         // [F][C][nv]
    Tout *out, *out2, *out3, *zero;   // [F][C][nv]; out2/out3/zero may be NULL
    double *partials_r;    // [F][part_stride] or NULL
    int part_stride;
};

template <typename Tin, typename Tout>
__global__ void __launch_bounds__(1024) k_project(ProjectArgs<Tin, Tout> a) {
    __shared__ double wred[32][3];
    __shared__ double coef[3];
    __shared__ double wsum[32];
    const int w = blockIdx.x, f = blockIdx.y, nv = a.g.nv, n = a.g.n;
    const size_t base = ((size_t)f * a.g.C + 2 * w) * nv;
    const int nr = a.g.n_remove[w];
    const double half_n = 0.5 * (n - 1);
    double t0 = 0, t1 = 0, t2 = 0;
    if (nr > 0)
        for (int e = threadIdx.x; e < 2 * nv; e += blockDim.x) {
            const int comp = e >= nv, i = e - comp * nv;
            const double v = (double)a.in[base + e];
            const double coord = ((comp ? a.g.iy[i] : a.g.ix[i]) - half_n) * a.g.d;
            if (comp) t1 += v; else t0 += v;
            t2 += coord * v;
        }
    t0 = warp_sum(t0); t1 = warp_sum(t1); t2 = warp_sum(t2);
    if ((threadIdx.x & 31) == 0) { wred[threadIdx.x >> 5][0] = t0; wred[threadIdx.x >> 5][1] = t1; wred[threadIdx.x >> 5][2] = t2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[3] = {0, 0, 0};
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { t[0] += wred[k][0]; t[1] += wred[k][1]; t[2] += wred[k][2]; }
        const double *G = a.g.Gs + w * 9;
        for (int u = 0; u < 3; ++u) {
            double s = 0.0;
            if (u < nr) for (int v = 0; v < nr; ++v) s += G[u * 3 + v] * t[v];
            coef[u] = s;
        }
    }
    __syncthreads();
    double rr = 0.0;
    for (int e = threadIdx.x; e < 2 * nv; e += blockDim.x) {
        const int comp = e >= nv, i = e - comp * nv;
        const double coord = ((comp ? a.g.iy[i] : a.g.ix[i]) - half_n) * a.g.d;
        const double v = (double)a.in[base + e] - (coef[comp] + coef[2] * coord);
        const Tout o = (Tout)v;
        a.out[base + e] = o;
        if (a.out2) a.out2[base + e] = o;
        if (a.out3) a.out3[base + e] = o;
        if (a.zero) a.zero[base + e] = (Tout)0;
        rr += (double)o * (double)o;
    }
    if (a.partials_r) {
        rr = warp_sum(rr);
        if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = rr;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += wsum[k];
            a.partials_r[(size_t)f * a.part_stride + w] = s;
        }
    }
}

// plain conversions between the fp32 ABI and the plan's arithmetic type
template <typename Tin, typename Tout>
__global__ void k_convert(const Tin *in, Tout *out, size_t count) {
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < count; e += (size_t)gridDim.x * blockDim.x)
        out[e] = (Tout)in[e];
}

// warm start (L428, L506): r = b - M q (q = W(Sigma_ss+Sigma_eta)W^T x0 from rows_inv), p = r, partial r.r
template <typename T>
__global__ void __launch_bounds__(256) k_warm_residual(UpdateArgs<T> a, const T *b, T *p_out) {
    __shared__ double red[32 * TOMO_NRED];
    __shared__ double coef[16 * 3];
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
    if (threadIdx.x == 0) mode_coeffs(a.g, red, coef);
    __syncthreads();
    const T half_n = (T)(0.5 * (a.g.n - 1));
    double rr = 0.0;
    const size_t base = (size_t)f * C * nv;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < C * nv; e += gridDim.x * blockDim.x) {
        const int c = e / nv, i = e - c * nv, w = c >> 1, comp = c & 1;
        const T coord = ((comp ? (T)a.g.iy[i] : (T)a.g.ix[i]) - half_n) * (T)a.g.d;
        const T qp = a.q[base + e] - ((T)coef[w * 3 + comp] + (T)coef[w * 3 + 2] * coord);
        const T rv = b[base + e] - qp;
        a.r[base + e] = rv;
        p_out[base + e] = rv;
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

// ------------------------------------------------------------------------------------------------ A7
// zeta~ along y for every (frame, channel, kx): Zs[f][kx][c][ky]
template <typename T> struct CosColsArgs {
    Stage<T> st;
    DevGeom g;
    int F;
    const typename cx_of<T>::type *T1;   // [F][C][Ph][n]
    typename cx_of<T>::type *Zs;         // [F][Ph][C][P]
};

template <typename T>
__global__ void __launch_bounds__(128) k_cos_cols_fwd(CosColsArgs<T> a) {
    typedef typename cx_of<T>::type C2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, n = a.g.n, C = a.g.C;
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NW = blockDim.x >> 5;
    C2 *A = tw + P + (size_t)warp * 2 * P, *B = A + P;
    load_twiddles<T>(tw, a.st);
    __syncthreads();
    const int items = a.F * C * Ph;
    for (int it = blockIdx.x * NW + warp; it < items; it += gridDim.x * NW) {
        const int f = it / (C * Ph), rem = it - f * C * Ph, c = rem / Ph, kx = rem - c * Ph;
        const C2 *src = a.T1 + (((size_t)f * C + c) * Ph + kx) * n;
        for (int i = lane; i < P; i += 32) A[i] = (i < n) ? src[i] : mk<T>((T)0, (T)0);
        C2 *Z = warp_fft<T, false>(A, B, a.st.fd, tw, lane);
        C2 *dst = a.Zs + (((size_t)f * Ph + kx) * C + c) * P;
        for (int i = lane; i < P; i += 32) dst[i] = Z[i];
        __syncwarp();
    }
}

// per (target, layer, kx): g~(ky) = sum_c xi~'(c, ky) zeta~_c(ky) for every frame of the chunk (the spectra are
// read from HBM once and reused from L1/L2 for the other frames), inverse FFT along y, keep rows y < n'.
template <typename T, typename S> struct CosMacArgs {
    Stage<T> st;
    DevGeom g;
    int F;
    const typename cx_of<T>::type *Zs;     // [F][Ph][C][P]
    const typename cx_of<S>::type *spec;   // [T][Kp][Ph][C][P]
    typename cx_of<T>::type *T2;           // [F][T][Kp][Ph][n']
};

template <typename T, typename S>
__global__ void __launch_bounds__(128) k_cos_mac_inv(CosMacArgs<T, S> a) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, C = a.g.C, np = a.g.n_p, TK = a.g.T * a.g.Kp;
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NW = blockDim.x >> 5;
    C2 *A = tw + P + (size_t)warp * 2 * P, *B = A + P;
    load_twiddles<T>(tw, a.st);
    __syncthreads();
    const int items = TK * Ph;
    for (int it = blockIdx.x * NW + warp; it < items; it += gridDim.x * NW) {
        const int tk = it / Ph, kx = it - tk * Ph;
        const S2 *sp = a.spec + ((size_t)tk * Ph + kx) * C * P;
        for (int f = 0; f < a.F; ++f) {
            const C2 *zs = a.Zs + ((size_t)f * Ph + kx) * C * P;
            for (int i = lane; i < P; i += 32) {
                T ar = (T)0, ai = (T)0;
                for (int c = 0; c < C; ++c) {
                    const S2 s = sp[(size_t)c * P + i];
                    const C2 z = zs[(size_t)c * P + i];
                    ar += (T)s.x * z.x - (T)s.y * z.y;
                    ai += (T)s.x * z.y + (T)s.y * z.x;
                }
                A[i] = mk<T>(ar, ai);
            }
            C2 *Z = warp_fft<T, true>(A, B, a.st.fd, tw, lane);
            C2 *dst = a.T2 + (((size_t)f * TK + tk) * Ph + kx) * np;
            for (int i = lane; i < np; i += 32) dst[i] = Z[i];
            __syncwarp();
        }
    }
}

// inverse FFT along x for row pairs of the n' x n' grid -> G[f][t][k][y][x]
template <typename T> struct CosRowsArgs {
    Stage<T> st;
    DevGeom g;
    int F;
    const typename cx_of<T>::type *T2;   // [F][T][Kp][Ph][n']
    T *G;                                // [F][T][Kp][n'][n']
};

template <typename T>
__global__ void __launch_bounds__(128) k_cos_rows_inv(CosRowsArgs<T> a) {
    typedef typename cx_of<T>::type C2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, np = a.g.n_p, TK = a.g.T * a.g.Kp, npr = (np + 1) / 2;
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NW = blockDim.x >> 5;
    C2 *A = tw + P + (size_t)warp * 2 * P, *B = A + P;
    load_twiddles<T>(tw, a.st);
    __syncthreads();
    const int items = a.F * TK * npr;
    for (int it = blockIdx.x * NW + warp; it < items; it += gridDim.x * NW) {
        const int ftk = it / npr, j = it - ftk * npr;
        const int y0 = 2 * j, y1 = 2 * j + 1;
        const bool two = y1 < np;
        const C2 *src = a.T2 + (size_t)ftk * Ph * np;
        for (int k = lane; k < Ph; k += 32) {
            const C2 u = src[(size_t)k * np + y0];
            const C2 v = two ? src[(size_t)k * np + y1] : mk<T>((T)0, (T)0);
            A[k] = mk<T>(u.x - v.y, u.y + v.x);
            if (k > 0 && 2 * k < P) A[P - k] = mk<T>(u.x + v.y, v.x - u.y);
        }
        C2 *Z = warp_fft<T, true>(A, B, a.st.fd, tw, lane);
        T *g0 = a.G + ((size_t)ftk * np + y0) * np;
        for (int x = lane; x < np; x += 32) {
            g0[x] = Z[x].x;
            if (two) g0[np + x] = Z[x].y;
        }
        __syncwarp();
    }
}

// phi[f][t][p] = sum_k sum_{4 taps} I'_k[p, tap] g_k[tap]   (Eq.16-17, Eq.32)
template <typename T>
__global__ void k_cos_gather(DevGeom g, int F, const T *G, const int *i0, const T *wt, T *phi) {
    // eight lanes per phase point, lane s takes the layers k = s, s + 8, ...; fixed-order (xor tree) sum
    const int np = g.n_p, n1 = g.n + 1, sub = threadIdx.x & 7;
    const size_t total = (size_t)F * g.T * g.nvp;
    const size_t stride = (size_t)gridDim.x * (blockDim.x >> 3);
    const size_t rounds = (total + stride - 1) / stride;
    size_t e = (size_t)blockIdx.x * (blockDim.x >> 3) + (threadIdx.x >> 3);
    for (size_t it = 0; it < rounds; ++it, e += stride) {
        T acc = (T)0;
        if (e < total) {
            const size_t ft = e / g.nvp;
            const int p = (int)(e - ft * g.nvp);
            const int px = g.pix[p], py = g.piy[p];
            for (int k = sub; k < g.Kp; k += 8) {
                const int ix0 = i0[k * n1 + px], iy0 = i0[k * n1 + py];
                const T wx = wt[k * n1 + px], wy = wt[k * n1 + py];
                const T *gk = G + ((ft * g.Kp + k) * np + iy0) * np + ix0;
                acc += ((T)1 - wy) * (((T)1 - wx) * gk[0] + wx * gk[1]) + wy * (((T)1 - wx) * gk[np] + wx * gk[np + 1]);
            }
        }
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (e < total && sub == 0) phi[e] = acc;
    }
}

// A8: phi_hat = M_phi W_phi phi: remove piston (always) and tip/tilt(/focus) over the valid phase points
// (Eq.35; Z_phi = [1, x, y, x^2+y^2], reading G14).  One CTA per (target, frame); fp32 out.
template <typename T>
__global__ void __launch_bounds__(1024) k_phase_project(DevGeom g, const T *phi, float *out) {
    __shared__ double wred[32][4];
    __shared__ double coef[4];
    const size_t base = ((size_t)blockIdx.y * g.T + blockIdx.x) * g.nvp;
    const int nc = 1 + g.n_remove_phase;
    const double half = 0.5 * g.n;
    double t[4] = {0, 0, 0, 0};
    for (int p = threadIdx.x; p < g.nvp; p += blockDim.x) {
        const double v = (double)phi[base + p];
        const double x = (g.pix[p] - half) * g.d, y = (g.piy[p] - half) * g.d;
        t[0] += v; t[1] += x * v; t[2] += y * v; t[3] += (x * x + y * y) * v;
    }
    for (int u = 0; u < 4; ++u) t[u] = warp_sum(t[u]);
    if ((threadIdx.x & 31) == 0) for (int u = 0; u < 4; ++u) wred[threadIdx.x >> 5][u] = t[u];
    __syncthreads();
    if (threadIdx.x == 0) {
        double s[4] = {0, 0, 0, 0};
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) for (int u = 0; u < 4; ++u) s[u] += wred[k][u];
        for (int u = 0; u < 4; ++u) {
            double c = 0.0;
            if (u < nc) for (int v = 0; v < nc; ++v) c += g.Gphi[u * 4 + v] * s[v];
            coef[u] = c;
        }
    }
    __syncthreads();
    for (int p = threadIdx.x; p < g.nvp; p += blockDim.x) {
        const double x = (g.pix[p] - half) * g.d, y = (g.piy[p] - half) * g.d;
        out[base + p] = (float)((double)phi[base + p] - (coef[0] + coef[1] * x + coef[2] * y + coef[3] * (x * x + y * y)));
    }
}

}  // namespace tomo
