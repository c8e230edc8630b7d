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

// (ar, ai) += (sx + i sy)(zx + i zy) with the contraction written out: k_cos_mac_inv and k_cos_mac_bulk round identically, so a frame
// of a batch (the former) equals its single-frame solve (the latter) bit for bit
__device__ __forceinline__ void cmac_acc(float &ar, float &ai, float sx, float sy, float zx, float zy) {
    ar = __fmaf_rn(sx, zx, ar); ar = __fmaf_rn(-sy, zy, ar); ai = __fmaf_rn(sx, zy, ai); ai = __fmaf_rn(sy, zx, ai);
}
__device__ __forceinline__ void cmac_acc(double &ar, double &ai, double sx, double sy, double zx, double zy) {
    ar = __fma_rn(sx, zx, ar); ar = __fma_rn(-sy, zy, ar); ai = __fma_rn(sx, zy, ai); ai = __fma_rn(sy, zx, ai);
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
                    cmac_acc(ar, ai, (T)s.x, (T)s.y, z.x, z.y);
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

// ---- bulk-copy variant of k_cos_mac_inv (one frame, fp32, P <= 256, C a compile-time constant).
// The kernel above keeps the streamed spectra in flight through registers: 36 warps per SM, each waiting on its own loads
// (long_scoreboard 64 % of the samples, 64 % of the HBM peak at cfg4).  Here the spectra of one (target, layer, k_x) item -- C P
// complex64, contiguous in HBM -- arrive by ONE bulk copy (`cp.async.bulk`, completion on an mbarrier) into a ring of stages
// shared by the whole CTA, so that the bytes in flight cost no registers and no warp has to wait for its own data:
//   * a CTA owns a contiguous range of items in [k_x][target, layer] order; thread ky < P keeps zeta~_c(k_x, ky), c < C, in
//     registers for as long as k_x stays the same;
//   * per item: wait for its stage, every thread forms g~(ky) = sum_c xi~'(c, ky) zeta~_c(ky) from shared memory and writes it to
//     one of NW small FFT buffers, the stage is refilled at once with the item NS ahead;
//   * every NW items the NW warps run one inverse y-FFT each and store rows y < n' (same warp_fft, same order of operations as
//     k_cos_mac_inv, see cmac_acc: the results are bitwise the same).
static const int kCosBulkThreads = 256;
static const int kCosBulkMaxStages = 8;

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// shared memory: ring[NS][CT P] | tw[P] | fb[NW][2][P] | full[NS]
static inline size_t cos_bulk_smem(int C, int P, int NS) {
    return ((size_t)NS * C * P + P + (size_t)(kCosBulkThreads / 32) * 2 * P) * 2 * sizeof(float) + (size_t)NS * 8;
}

template <int CT>
__global__ void __launch_bounds__(kCosBulkThreads, 2) k_cos_mac_bulk(CosMacArgs<float, float> a, int NS) {
    typedef float2 C2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, np = a.g.n_p, TK = a.g.T * a.g.Kp;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int NW = kCosBulkThreads / 32;
    const size_t stage = (size_t)CT * P;
    C2 *ring = reinterpret_cast<C2 *>(smem_raw);
    C2 *tw = ring + (size_t)NS * stage;
    C2 *fb = tw + P;
    unsigned long long *full = reinterpret_cast<unsigned long long *>(fb + (size_t)NW * 2 * P);
    const unsigned bytes = (unsigned)(stage * sizeof(C2));
    // this CTA's items e in [e0, e1), e = kx TK + tk
    const int total = Ph * TK, per = (total + gridDim.x - 1) / gridDim.x;
    const int e0 = min(total, (int)blockIdx.x * per), e1 = min(total, e0 + per), n_my = e1 - e0;
    auto src_of = [&](int e) { const int kx = e / TK, tk = e - kx * TK; return a.spec + ((size_t)tk * Ph + kx) * stage; };
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(full + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    load_twiddles<float>(tw, a.st);
    __syncthreads();
    if (tid == 0)
        for (int s = 0; s < NS && s < n_my; ++s) { mbar_expect_tx(full + s, bytes); bulk_g2s(ring + (size_t)s * stage, src_of(e0 + s), bytes, full + s); }
    C2 z[CT];
    int kx_cur = -1;
#pragma unroll 1
    for (int i = 0; i < n_my; ++i) {
        const int e = e0 + i, kx = e / TK, tk = e - kx * TK, s = i % NS, j = i % NW;
        if (kx != kx_cur) {
            kx_cur = kx;
            if (tid < P) {
#pragma unroll
                for (int c = 0; c < CT; ++c) z[c] = a.Zs[((size_t)kx * CT + c) * P + tid];
            }
        }
        mbar_wait(full + s, (unsigned)((i / NS) & 1));
        if (tid < P) {
            const C2 *sp = ring + (size_t)s * stage + tid;
            float ar = 0.f, ai = 0.f;
#pragma unroll
            for (int c = 0; c < CT; ++c) {
                const C2 v = sp[(size_t)c * P];
                cmac_acc(ar, ai, v.x, v.y, z[c].x, z[c].y);
            }
            fb[(size_t)j * 2 * P + tid] = make_float2(ar, ai);
        }
        __syncthreads();                                    // the stage has been read by everyone, fb[j] is complete
        if (tid == 0 && i + NS < n_my) { mbar_expect_tx(full + s, bytes); bulk_g2s(ring + (size_t)s * stage, src_of(e + NS), bytes, full + s); }
        if (j == NW - 1 || i == n_my - 1) {
            if (warp <= j) {
                const int ei = e - j + warp, kxi = ei / TK, tki = ei - kxi * TK;
                C2 *A = fb + (size_t)warp * 2 * P;
                C2 *Z = warp_fft<float, true>(A, A + P, a.st.fd, tw, lane);
                C2 *dst = a.T2 + ((size_t)tki * Ph + kxi) * np;
                for (int y = lane; y < np; y += 32) dst[y] = Z[y];
            }
            __syncthreads();                                // before the next group overwrites the FFT buffers
        }
        (void)tk;
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
