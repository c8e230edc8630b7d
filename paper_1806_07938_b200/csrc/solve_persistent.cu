// solve_persistent.cu -- persistent cooperative CG solver: ONE kernel per solve, two grid barriers per iteration.
//
// The textbook CG recurrences (PAPER.md S2.G L337, Eq.12; oracle/solver.py) are kept, but the work is
// re-ordered so that an iteration has only the two all-to-all exchanges the 2-D FFT itself needs:
//
//   phase C_k (one CTA per k_x slab, all channels):   rho_k, beta_k from the r.r partials;
//        p~rows_k = r~rows_k + beta_k p~rows_{k-1}    (the x-FFT is linear, so p = r + beta p is formed in the
//                                                      half-transformed domain; p~rows stays with its slab)
//        y-FFT, per-frequency C x C block product with the Hermitian-packed kernel spectra pinned in shared
//        memory (Eq.22, Eq.30), + sigma^2 p~ (Sigma_eta, L260), inverse y-FFT -> T2
//        p.q and the modal sums Z^T q (Eq.36) by Parseval from p~, y~ and the mask spectra
//   ---- grid barrier B ----
//   phase R_k (one warp per (channel, row pair)):      alpha_k = rho_k / p.q, mode coefficients;
//        inverse x-FFT, crop + mask (S_2, W_s; Eq.24-27, Eq.34), q' = M_s q,
//        p_k = r_k + beta_k p_{k-1} (spatial copy), x += alpha p, r -= alpha q', partial r.r,
//        forward x-FFT of the NEW residual rows (S_1, Eq.18-21) -> T1
//   ---- grid barrier A ----
//
// p.q is taken in the frequency domain (Parseval; p is zero outside the pupil, so the crop does not matter and
// p.M_s q = p.q for p in range(M_s)); every reduction is a fixed-order two-stage sum with fp64 scalars, so a
// fixed-count solve is bit-reproducible.  Sigma_eta must be uniform per channel here (all configs); otherwise the
// caller falls back to the multi-kernel solver.
#include <algorithm>
#include <complex>
#include <cstring>
#include <string>
#include <vector>

#include "tomo.h"
#include "tomo_kernels.cuh"
#include "tomo_kernels_cos.cuh"
#include "tomo_plan.hpp"

namespace tomo {

static const int kPThreads = 512;
static const int kPWarps = kPThreads / 32;

enum { PM_COLD = 0, PM_WARM = 1, PM_STATE = 2 };
enum { PT_START = 0, PT_RHO = 1, PT_BUILD = 2, PT_FFT = 3, PT_MAC = 4, PT_INV = 5, PT_BAR_B = 6, PT_SCAL = 7, PT_ROWS = 8, PT_BAR_A = 9, PT_N = 10 };

// per-frame scalar block in shared memory (doubles)
enum { SC_RHO = 0, SC_RHO_PREV = 1, SC_BETA = 2, SC_ALPHA = 3, SC_UPD = 4, SC_PQ = 5, SC_HEAD = 6 };

template <typename T, typename S> struct PArgs {
    Stage<T> st;
    DevGeom g;
    int F, n_iter, mode, finalize_p;
    int G;                       // grid size (CTAs)
    int npad;                    // 2 * npairs
    int U;                       // row units per frame = C * npairs
    int NQ;                      // slab partial quantities: 1 + C (+ C with focus removal)
    int nq_m;                    // mask spectra: 1 (mask) or 3 (mask, x-weighted, y-weighted)
    int SB;                      // doubles per frame in the scalar block
    int spec_smem;               // kernel spectra slice pinned in shared memory
    int vec_smem;                // x, r, p rows of the CTA's units held in shared memory for the whole solve
    int any_remove;
    // shared-memory layout (byte offsets)
    int off_ms, off_work, off_scal, off_wred, off_tab, off_upart, off_rowptr, off_ix, off_vec, off_spec, wred_stride;
    const float *s_in;           // [F][C][nv] slopes (COLD/WARM)
    const float *x0;             // [F][C][nv] warm start (WARM)
    T *x, *r, *p, *b;            // [F][C][nv]
    typename cx_of<T>::type *T1;    // [F][Ph][C][npad]     x-FFT of the current residual rows
    typename cx_of<T>::type *T1p;   // [F][Ph][C][npad]     x-FFT of the search direction (slab-private state)
    typename cx_of<T>::type *T2;    // [F][C][npairs][Ph][2]
    const typename cx_of<S>::type *spec;   // [Ph][n_pair][P]
    int n_pair;
    const typename cx_of<T>::type *mspec;  // [nq_m][Ph][P]  spectra of the pupil mask (and coordinate-weighted masks)
    const T *s2c;                // [C] sigma^2_c / P^2
    double *part_r;              // [F][G]       r.r per CTA
    double *part_s;              // [F][NQ][Ph]  per slab: p.q, sum q_c, sum coord q_c
    double *part_i;              // [F][U][2]    init: sum s, sum coord s per row unit
    double *hist;                // [F][hist_stride] rho_k
    int hist_stride;
    double *alpha;               // [F]
    double *scal_out;            // [3] rho_{k+1}, alpha, beta (finalize_p, frame 0) or NULL
    unsigned *flags;             // [G] epoch each CTA has completed (grid barrier)
    long long *dbg;              // [G][n_iter][PT_N] clock64 stamps of thread 0 (measurement aid) or NULL
};

// ---- grid barrier: one arrival counter (measured on B200: ~2400 cycles for 16..148 CTAs; per-CTA flag arrays polled by
// every CTA hot-spot one L2 slice and cost 2-3x more).  Writers: data stores -> bar.sync -> thread 0: red.release.
// Readers: thread 0 ld.acquire until all arrived -> bar.sync -> L2 (.cg) loads of the exchanged data.
__device__ __forceinline__ void grid_sync(unsigned *ctr, unsigned target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
        unsigned v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
        } while ((int)(v - target) < 0);
    }
    __syncthreads();
}

template <typename T> __device__ __forceinline__ double div_as(double a, double b) { return (double)((T)a / (T)b); }

__device__ __forceinline__ float warp_sum_t(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum_t(double v) { return warp_sum(v); }

// deterministic sum by one warp of up to 160 contiguous doubles other CTAs wrote: all loads in flight at once
__device__ __forceinline__ double warp_sum_cg160(const double *src, int count, int lane) {
    double v[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) { const int i = lane + 32 * m; v[m] = (i < count) ? __ldcg(src + i) : 0.0; }
    return warp_sum(((v[0] + v[1]) + (v[2] + v[3])) + v[4]);
}
__device__ __forceinline__ double warp_sum_cg(const double *src, int count, int stride, int lane) {
    double s = 0.0;
    for (int i = lane; i < count; i += 32) s += __ldcg(src + (size_t)i * stride);
    return warp_sum(s);
}

// two adjacent complex values (16-byte aligned for fp32) through L2
__device__ __forceinline__ void ldcg_pair(const float2 *p, float2 &u, float2 &v) {
    const float4 t = __ldcg(reinterpret_cast<const float4 *>(p));
    u = make_float2(t.x, t.y); v = make_float2(t.z, t.w);
}
__device__ __forceinline__ void ldcg_pair(const double2 *p, double2 &u, double2 &v) { u = __ldcg(p); v = __ldcg(p + 1); }
__device__ __forceinline__ void ld_pair(const float2 *p, float2 &u, float2 &v) {
    const float4 t = *reinterpret_cast<const float4 *>(p);
    u = make_float2(t.x, t.y); v = make_float2(t.z, t.w);
}
__device__ __forceinline__ void ld_pair(const double2 *p, double2 &u, double2 &v) { u = p[0]; v = p[1]; }
__device__ __forceinline__ void st_pair(float2 *p, float2 u, float2 v) { *reinterpret_cast<float4 *>(p) = make_float4(u.x, u.y, v.x, v.y); }
__device__ __forceinline__ void st_pair(double2 *p, double2 u, double2 v) { p[0] = u; p[1] = v; }

// ---- FFT dispatch: compile-time plans for the sizes the configs use (fp32), run-time plan otherwise
template <typename T, bool INV, int P>
__device__ __noinline__ typename cx_of<T>::type *wfft_s(typename cx_of<T>::type *a, typename cx_of<T>::type *b,
                                                        const typename cx_of<T>::type *tw, int lane) {
    return warp_fft_static<T, INV, P>(a, b, tw, lane);
}
template <typename T, bool INV>
__device__ __noinline__ typename cx_of<T>::type *wfft_generic(typename cx_of<T>::type *a, typename cx_of<T>::type *b, const FftDesc &fd,
                                                              const typename cx_of<T>::type *tw, int lane) {
    return warp_fft<T, INV>(a, b, fd, tw, lane);
}
template <typename T, bool INV>
__device__ __forceinline__ typename cx_of<T>::type *wfft(typename cx_of<T>::type *a, typename cx_of<T>::type *b, const FftDesc &fd,
                                                         const typename cx_of<T>::type *tw, int lane) {
    if constexpr (sizeof(T) == 4) {
        switch (fd.P) {
            case 16: return wfft_s<T, INV, 16>(a, b, tw, lane);
            case 20: return wfft_s<T, INV, 20>(a, b, tw, lane);
            case 24: return wfft_s<T, INV, 24>(a, b, tw, lane);
            case 32: return wfft_s<T, INV, 32>(a, b, tw, lane);
            case 40: return wfft_s<T, INV, 40>(a, b, tw, lane);
            case 64: return wfft_s<T, INV, 64>(a, b, tw, lane);
            case 128: return wfft_s<T, INV, 128>(a, b, tw, lane);
            case 160: return wfft_s<T, INV, 160>(a, b, tw, lane);
            case 192: return wfft_s<T, INV, 192>(a, b, tw, lane);
            case 256: return wfft_s<T, INV, 256>(a, b, tw, lane);
            default: break;
        }
    }
    return wfft_generic<T, INV>(a, b, fd, tw, lane);
}

// ---- per-frequency block product of one k_x slab (Eq.22, Eq.30) + Sigma_eta (L260) + Parseval partials.
// Warps are grouped: WPG = ceil(P/32) warps cover the k_y range, group g owns a contiguous range of output channels.
// CT > 0: the C inputs of this k_y are held in registers (compile-time channel count); CT = 0: read from shared memory.
template <typename T, typename S, int CT>
__device__ __noinline__ void mac_slab(const typename cx_of<T>::type *X, typename cx_of<T>::type *Y,
                                      const typename cx_of<S>::type *spec, const typename cx_of<T>::type *ms, const T *s2c,
                                      int C, int P, int nq_m, int any_remove, double *wred, int wred_stride, int warp, int lane) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    const int WPG = (P + 31) >> 5;
    const int Goc = min(kPWarps / WPG, C);
    const int grp = warp / WPG, ky = (warp - grp * WPG) * 32 + lane;
    if (grp >= Goc) return;
    const int oc_lo = grp * C / Goc, oc_hi = (grp + 1) * C / Goc;
    const bool act = ky < P;
    const int kyc = act ? ky : 0;
    C2 x[CT > 0 ? CT : 1];
    if (CT > 0) {
#pragma unroll
        for (int ci = 0; ci < CT; ++ci) x[ci] = X[(size_t)ci * P + kyc];
    }
    C2 m0 = mk<T>((T)0, (T)0), m1 = m0, m2 = m0;
    if (any_remove) { m0 = ms[kyc]; if (nq_m > 1) { m1 = ms[P + kyc]; m2 = ms[2 * P + kyc]; } }
    T pap = (T)0;
    for (int oc = oc_lo; oc < oc_hi; ++oc) {
        const C2 xo = X[(size_t)oc * P + kyc];
        const T s2 = s2c[oc];
        T ar = s2 * xo.x, ai = s2 * xo.y;
        const S2 *sp = spec + kyc;
        const int base_oc = oc * C - (oc * (oc - 1)) / 2;      // pair (oc, oc)
        int idx = oc;                                           // pair (0, oc)
        if (CT > 0) {
#pragma unroll
            for (int ci = 0; ci < CT; ++ci) {
                const bool lower = ci < oc;
                const S2 s = sp[(size_t)(lower ? idx : base_oc + ci - oc) * P];
                const T sr = (T)s.x, si = lower ? -(T)s.y : (T)s.y;
                ar += sr * x[ci].x - si * x[ci].y;
                ai += sr * x[ci].y + si * x[ci].x;
                idx += C - ci - 1;
            }
        } else {
            for (int ci = 0; ci < C; ++ci) {
                const bool lower = ci < oc;
                const S2 s = sp[(size_t)(lower ? idx : base_oc + ci - oc) * P];
                const C2 xv = X[(size_t)ci * P + kyc];
                const T sr = (T)s.x, si = lower ? -(T)s.y : (T)s.y;
                ar += sr * xv.x - si * xv.y;
                ai += sr * xv.y + si * xv.x;
                idx += C - ci - 1;
            }
        }
        if (!act) { ar = (T)0; ai = (T)0; }
        else Y[(size_t)oc * P + ky] = mk<T>(ar, ai);
        pap += xo.x * ar + xo.y * ai;                           // Re(conj(p~) y~)
        if (any_remove) {
            T sq = m0.x * ar + m0.y * ai, fq = (T)0;            // Re(conj(m~) y~)
            sq = warp_sum_t(sq);
            if (nq_m > 1) { const C2 mm = (oc & 1) ? m2 : m1; fq = warp_sum_t(mm.x * ar + mm.y * ai); }
            if (lane == 0) {
                wred[warp * wred_stride + 1 + 2 * (oc - oc_lo)] = (double)sq;
                wred[warp * wred_stride + 2 + 2 * (oc - oc_lo)] = (double)fq;
            }
        }
    }
    pap = warp_sum_t(pap);
    if (lane == 0) wred[warp * wred_stride] = (double)pap;
}

template <typename T, typename S>
__global__ void __launch_bounds__(kPThreads, 1) k_persistent(PArgs<T, S> a) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.st.P, Ph = a.st.Ph, n = a.g.n, nv = a.g.nv, C = a.g.C, npairs = a.g.npairs, N = a.g.N;
    const int F = a.F, U = a.U, NQ = a.NQ, SB = a.SB, G = a.G, npad = a.npad;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, NW = kPWarps, b = blockIdx.x;
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    C2 *ms = reinterpret_cast<C2 *>(smem_raw + a.off_ms);
    C2 *work = reinterpret_cast<C2 *>(smem_raw + a.off_work);
    double *scal = reinterpret_cast<double *>(smem_raw + a.off_scal);
    double *wred = reinterpret_cast<double *>(smem_raw + a.off_wred);
    double *sGs = reinterpret_cast<double *>(smem_raw + a.off_tab);
    int *s_nrem = reinterpret_cast<int *>(sGs + 9 * N);
    T *s_s2c = reinterpret_cast<T *>(s_nrem + N + (N & 1));
    FftDesc *sfd = reinterpret_cast<FftDesc *>(s_s2c + C + (C & 1) * (sizeof(T) == 4));
    double *upart = reinterpret_cast<double *>(smem_raw + a.off_upart);
    int *s_rowptr = reinterpret_cast<int *>(smem_raw + a.off_rowptr);
    unsigned short *s_ix = reinterpret_cast<unsigned short *>(smem_raw + a.off_ix);
    T *svec = reinterpret_cast<T *>(smem_raw + a.off_vec);
    S2 *sspec = reinterpret_cast<S2 *>(smem_raw + a.off_spec);
    unsigned epoch = 0;
    const T half_n = (T)(0.5 * (n - 1)), dd = (T)a.g.d;
    int k = -2;                                      // iteration index seen by PSTAMP (no stamps outside the loop)
#define PSTAMP(pt) do { if (a.dbg && tid == 0 && k >= 0) a.dbg[((size_t)b * a.n_iter + k) * PT_N + (pt)] = clock64(); } while (0)
#define GRID_SYNC() do { epoch += G; grid_sync(a.flags, epoch); } while (0)

    // ---- slab ownership: CTA b owns k_x = b % Ph and a contiguous share of the frames
    const int kx = b % Ph;
    int f_lo, f_hi;
    {
        const int cnt = (G - 1 - kx) / Ph + 1, rk = b / Ph;
        f_lo = (int)((long long)rk * F / cnt);
        f_hi = (int)((long long)(rk + 1) * F / cnt);
        if (F == 1) { f_lo = 0; f_hi = (rk == 0) ? 1 : 0; }
    }
    const bool has_slab = f_hi > f_lo;
    const S2 *gspec = a.spec + (size_t)kx * a.n_pair * P;
    const T wkx = (kx == 0 || 2 * kx == P) ? (T)1 : (T)2;
    // ---- row units of this CTA: ut = b + i G, i < nu; unit i is processed by warp NW-1 - (i % NW)
    const int nu = (b < F * U) ? (F * U - b + G - 1) / G : 0;
    const int i_first = NW - 1 - warp;

    load_twiddles<T>(tw, a.st);
    for (int i = tid; i <= n; i += kPThreads) s_rowptr[i] = a.g.row_ptr[i];
    for (int i = tid; i < nv; i += kPThreads) s_ix[i] = (unsigned short)a.g.ix[i];
    for (int i = tid; i < 9 * N; i += kPThreads) sGs[i] = a.g.Gs[i];
    for (int i = tid; i < N; i += kPThreads) s_nrem[i] = a.g.n_remove[i];
    for (int i = tid; i < C; i += kPThreads) s_s2c[i] = a.s2c[i];
    if (tid == 0) *sfd = a.st.fd;
    if (has_slab) {
        for (int q = 0; q < a.nq_m; ++q)
            for (int i = tid; i < P; i += kPThreads) ms[q * P + i] = a.mspec[((size_t)q * Ph + kx) * P + i];
        if (a.spec_smem)
            for (int i = tid; i < a.n_pair * P; i += kPThreads) sspec[i] = gspec[i];
    }
    for (int i = tid; i < F * SB; i += kPThreads) scal[i] = 0.0;
    __syncthreads();
    const S2 *spec = a.spec_smem ? sspec : gspec;

    // per-WFS mode coefficients (Z^T Z)^-1 Z^T q from the channel sums (Eq.36): thread t -> (frame, WFS)
    auto mode_coefs = [&](int t) {
        const int f = t / N, i = t - f * N;
        double *sc = scal + f * SB;
        const double *S0 = sc + SC_HEAD, *S1 = sc + SC_HEAD + C;
        const double tq[3] = {S0[2 * i], S0[2 * i + 1], S1[2 * i] + S1[2 * i + 1]};
        const int nr = s_nrem[i];
        for (int u = 0; u < 3; ++u) {
            double s = 0.0;
            if (u < nr) for (int v = 0; v < nr; ++v) s += sGs[i * 9 + u * 3 + v] * tq[v];
            sc[SC_HEAD + 2 * C + i * 3 + u] = s;
        }
    };

    struct Unit { int f, u, c, j, comp, w, y0, s0, s1, len; bool two; size_t base; };
    auto unit_of = [&](int i) {
        Unit q;
        const int ut = b + i * G;
        q.f = ut / U; q.u = ut - q.f * U; q.c = q.u / npairs; q.j = q.u - q.c * npairs; q.comp = q.c & 1; q.w = q.c >> 1;
        q.y0 = 2 * q.j; q.two = q.y0 + 1 < n;
        q.s0 = s_rowptr[q.y0]; q.s1 = s_rowptr[q.y0 + 1]; q.len = s_rowptr[min(q.y0 + 2, n)] - q.s0;
        q.base = ((size_t)q.f * C + q.c) * nv + q.s0;
        return q;
    };
    // x, r, p of unit i, element e = valid index - s0
    auto vec_x = [&](int i, const Unit &q) { return a.vec_smem ? svec + (size_t)i * 6 * n : a.x + q.base; };
    auto vec_r = [&](int i, const Unit &q) { return a.vec_smem ? svec + (size_t)i * 6 * n + 2 * n : a.r + q.base; };
    auto vec_p = [&](int i, const Unit &q) { return a.vec_smem ? svec + (size_t)i * 6 * n + 4 * n : a.p + q.base; };

    C2 *bufA = work + (size_t)warp * 2 * P, *bufB = bufA + P;

    // forward x-FFT of two rows held as (.x = row y0, .y = row y1) in `in`, split into the two half-spectra -> T1
    auto fwd_rows_to_T1 = [&](C2 *in, C2 *other, const Unit &q) {
        C2 *Z = wfft<T, false>(in, other, *sfd, tw, lane);
        C2 *out = a.T1 + (((size_t)q.f * Ph) * C + q.c) * npad + q.y0;
#pragma unroll
        for (int m = 0; m < 5; ++m) {
            const int kk = lane + 32 * m;
            if (kk < Ph) {
                const C2 z1 = Z[kk], z2 = Z[kk == 0 ? 0 : P - kk];
                st_pair(out + (size_t)kk * C * npad, mk<T>((T)0.5 * (z1.x + z2.x), (T)0.5 * (z1.y - z2.y)),
                        q.two ? mk<T>((T)0.5 * (z1.y + z2.y), (T)-0.5 * (z1.x - z2.x)) : mk<T>((T)0, (T)0));
            }
        }
        __syncwarp();
    };
    // r.r of the CTA's units, per frame, in unit order -> part_r[f][b]
    auto publish_rr = [&]() {
        __syncthreads();
        for (int f = tid; f < F; f += kPThreads) {
            double s = 0.0;
            for (int i = 0; i < nu; ++i) if ((b + i * G) / U == f) s += upart[i];
            a.part_r[(size_t)f * G + b] = s;
        }
    };

    // ================================================================ init (A1: b = M_s s, Eq.33-34)
    if (a.mode != PM_STATE) {
        if (a.any_remove) {
            for (int i = i_first; i < nu; i += NW) {
                const Unit q = unit_of(i);
                const float *sv = a.s_in + q.base;
                double t0 = 0.0, t1 = 0.0;
                for (int e = lane; e < q.len; e += 32) {
                    const int ii = q.s0 + e, y = (ii >= q.s1) ? q.y0 + 1 : q.y0;
                    const double v = (double)sv[e];
                    const double coord = ((q.comp ? y : (int)s_ix[ii]) - 0.5 * (n - 1)) * a.g.d;
                    t0 += v; t1 += coord * v;
                }
                t0 = warp_sum(t0); t1 = warp_sum(t1);
                if (lane == 0) { a.part_i[((size_t)q.f * U + q.u) * 2] = t0; a.part_i[((size_t)q.f * U + q.u) * 2 + 1] = t1; }
            }
            GRID_SYNC();
            for (int item = warp; item < F * C * 2; item += NW) {
                const int f = item / (2 * C), rem = item - f * 2 * C, e = rem / C, c = rem - e * C;
                const double s = warp_sum_cg(a.part_i + ((size_t)f * U + c * npairs) * 2 + e, npairs, 2, lane);
                if (lane == 0) scal[f * SB + SC_HEAD + rem] = s;
            }
            __syncthreads();
            for (int t = tid; t < F * N; t += kPThreads) mode_coefs(t);
            __syncthreads();
        }
        // b = s - Z a ; cold: x = 0, r = p = b ; warm: x = x0, FFT input = x0
        for (int i = i_first; i < nu; i += NW) {
            const Unit q = unit_of(i);
            const double *coef = scal + q.f * SB + SC_HEAD + 2 * C + q.w * 3;
            T *ux = vec_x(i, q), *ur = vec_r(i, q), *up = vec_p(i, q);
            for (int e = lane; e < P; e += 32) bufA[e] = mk<T>((T)0, (T)0);
            __syncwarp();
            double rr = 0.0;
            for (int e = lane; e < q.len; e += 32) {
                const int ii = q.s0 + e;
                const bool row1 = ii >= q.s1;
                const int xc = s_ix[ii], y = row1 ? q.y0 + 1 : q.y0;
                const double coord = ((q.comp ? y : xc) - 0.5 * (n - 1)) * a.g.d;
                const T bv = (T)((double)a.s_in[q.base + e] - (coef[q.comp] + coef[2] * coord));
                T fv = bv;
                if (a.mode == PM_WARM) {
                    const T xv = (T)a.x0[q.base + e];
                    a.b[q.base + e] = bv; ux[e] = xv; fv = xv;
                } else {
                    ux[e] = (T)0; ur[e] = bv; up[e] = bv;
                    rr += (double)bv * (double)bv;
                }
                if (row1) bufA[xc].y = fv; else bufA[xc].x = fv;
            }
            rr = warp_sum(rr);
            if (lane == 0) upart[i] = rr;
            fwd_rows_to_T1(bufA, bufB, q);
        }
    } else {
        // STATE: x, r, p, rho_0 given; FFT of the p rows
        for (int i = i_first; i < nu; i += NW) {
            const Unit q = unit_of(i);
            T *ux = vec_x(i, q), *ur = vec_r(i, q), *up = vec_p(i, q);
            for (int e = lane; e < P; e += 32) bufA[e] = mk<T>((T)0, (T)0);
            __syncwarp();
            for (int e = lane; e < q.len; e += 32) {
                const int ii = q.s0 + e, xc = s_ix[ii];
                const T pv = a.p[q.base + e];
                if (a.vec_smem) { ux[e] = a.x[q.base + e]; ur[e] = a.r[q.base + e]; up[e] = pv; }
                if (ii >= q.s1) bufA[xc].y = pv; else bufA[xc].x = pv;
            }
            if (lane == 0) upart[i] = 0.0;
            fwd_rows_to_T1(bufA, bufB, q);
        }
    }
    publish_rr();
    GRID_SYNC();

    // ================================================================ iterations (k = -1 is the warm-start product A x0)
    const int k_begin = (a.mode == PM_WARM) ? -1 : 0;
    const bool res_in_A = (a.st.fd.nrad & 1) == 0;     // FFT result lands in its first argument iff nrad is even
    const int n_t1 = C * npairs;                        // complex pairs in one T1 slab
    for (k = k_begin; k < a.n_iter; ++k) {
        const bool pre = k < 0;
        const bool take_new = pre || k == 0;            // p~ = T1 (p_0, or x0 for the warm-start product)
        PSTAMP(PT_START);
        // ---------------------------------------------------------- phase C: slab (kx, f)
        C2 n0[2], n1[2], o0[2], o1[2];
        auto prefetch_slab = [&](int f, bool with_old) {
            const C2 *t1 = a.T1 + ((size_t)f * Ph + kx) * C * npad;
            const C2 *t1p = a.T1p + ((size_t)f * Ph + kx) * C * npad;
#pragma unroll
            for (int m = 0; m < 2; ++m) {
                const int e2 = tid + m * kPThreads;
                if (e2 < n_t1) {
                    ldcg_pair(t1 + 2 * e2, n0[m], n1[m]);
                    if (with_old) ld_pair(t1p + 2 * e2, o0[m], o1[m]);
                }
            }
        };
        if (has_slab) prefetch_slab(f_lo, !take_new);
        // scalars: rho_k, beta_k
        if (!pre) {
            for (int f = warp; f < F; f += NW) {
                double rho;
                if (k == 0 && a.mode == PM_STATE) rho = a.hist[(size_t)f * a.hist_stride];
                else rho = warp_sum_cg160(a.part_r + (size_t)f * G, G, lane);
                if (lane == 0) {
                    double *sc = scal + f * SB;
                    const double rho_prev = sc[SC_RHO];
                    const bool upd = (k > 0) && (sc[SC_ALPHA] != 0.0) && (rho_prev > 0.0);
                    sc[SC_RHO_PREV] = rho_prev;
                    sc[SC_RHO] = rho;
                    sc[SC_BETA] = upd ? div_as<T>(rho, rho_prev) : 0.0;
                    sc[SC_UPD] = upd ? 1.0 : 0.0;
                    if (b == 0) a.hist[(size_t)f * a.hist_stride + k] = rho;
                }
            }
        }
        __syncthreads();
        PSTAMP(PT_RHO);
        for (int f = f_lo; f < f_hi; ++f) {
            const double *sc = scal + f * SB;
            const bool upd = !pre && sc[SC_UPD] != 0.0;
            const T beta = (T)sc[SC_BETA];
            C2 *Ubuf = work, *Vbuf = work + (size_t)C * P;
            C2 *t1p = a.T1p + ((size_t)f * Ph + kx) * C * npad;
            if (f != f_lo) prefetch_slab(f, !take_new);
            // zero padding rows n..P-1, then p~rows = r~rows + beta p~rows_old on rows 0..n-1
            for (int e = tid; e < C * (P - n); e += kPThreads) { const int c = e / (P - n), y = n + e - c * (P - n); Ubuf[c * P + y] = mk<T>((T)0, (T)0); }
#pragma unroll
            for (int m = 0; m < 2; ++m) {
                const int e2 = tid + m * kPThreads;
                if (e2 < n_t1) {
                    C2 v0, v1;
                    if (take_new) { v0 = n0[m]; v1 = n1[m]; }
                    else if (upd) { v0 = mk<T>(n0[m].x + beta * o0[m].x, n0[m].y + beta * o0[m].y); v1 = mk<T>(n1[m].x + beta * o1[m].x, n1[m].y + beta * o1[m].y); }
                    else { v0 = o0[m]; v1 = o1[m]; }
                    if (take_new || upd) st_pair(t1p + 2 * e2, v0, v1);
                    const int c = e2 / npairs, y = 2 * (e2 - c * npairs);
                    Ubuf[c * P + y] = v0;
                    if (y + 1 < n) Ubuf[c * P + y + 1] = v1;
                }
            }
            __syncthreads();
            PSTAMP(PT_BUILD);
            for (int c = warp; c < C; c += NW) wfft<T, false>(Ubuf + (size_t)c * P, Vbuf + (size_t)c * P, *sfd, tw, lane);
            __syncthreads();
            C2 *X = res_in_A ? Ubuf : Vbuf, *Y = res_in_A ? Vbuf : Ubuf;
            PSTAMP(PT_FFT);
            switch (C) {
                case 4: mac_slab<T, S, 4>(X, Y, spec, ms, s_s2c, C, P, a.nq_m, a.any_remove, wred, a.wred_stride, warp, lane); break;
                case 6: mac_slab<T, S, 6>(X, Y, spec, ms, s_s2c, C, P, a.nq_m, a.any_remove, wred, a.wred_stride, warp, lane); break;
                case 8: mac_slab<T, S, 8>(X, Y, spec, ms, s_s2c, C, P, a.nq_m, a.any_remove, wred, a.wred_stride, warp, lane); break;
                case 12: mac_slab<T, S, 12>(X, Y, spec, ms, s_s2c, C, P, a.nq_m, a.any_remove, wred, a.wred_stride, warp, lane); break;
                case 16: mac_slab<T, S, 16>(X, Y, spec, ms, s_s2c, C, P, a.nq_m, a.any_remove, wred, a.wred_stride, warp, lane); break;
                default: mac_slab<T, S, 0>(X, Y, spec, ms, s_s2c, C, P, a.nq_m, a.any_remove, wred, a.wred_stride, warp, lane); break;
            }
            __syncthreads();
            PSTAMP(PT_MAC);
            // slab partials (fixed order) and the inverse y-FFTs
            const int tq = tid - (kPThreads - 64);          // the last two warps: no (or the last) y-FFT channels
            if (tq >= 0 && tq < NQ) {
                const int WPG = (P + 31) >> 5, Goc = min(NW / WPG, C);
                int w0 = 0, w1 = Goc * WPG, off = 0;
                if (tq > 0) {
                    const int e = (tq - 1) / C, oc = (tq - 1) - e * C;
                    int g2 = 0;
                    while ((g2 + 1) * C / Goc <= oc) ++g2;
                    w0 = g2 * WPG; w1 = w0 + WPG; off = 1 + 2 * (oc - g2 * C / Goc) + e;
                }
                double s = 0.0;
                if (tq == 0 || a.any_remove) {
#pragma unroll
                    for (int w = 0; w < kPWarps; ++w) { const int ww = w0 + w; if (ww < w1) s += wred[ww * a.wred_stride + off]; }
                }
                a.part_s[((size_t)f * NQ + tq) * Ph + kx] = (double)wkx * s;
            }
            for (int c = warp; c < C; c += NW) {
                C2 *res = wfft<T, true>(Y + (size_t)c * P, X + (size_t)c * P, *sfd, tw, lane);
                C2 *dst = a.T2 + ((size_t)f * C + c) * npairs * Ph * 2 + (size_t)kx * 2;
                for (int j = lane; j < npairs; j += 32)
                    st_pair(dst + (size_t)j * Ph * 2, res[2 * j], (2 * j + 1 < n) ? res[2 * j + 1] : mk<T>((T)0, (T)0));
            }
            __syncthreads();
        }
        PSTAMP(PT_INV);
        GRID_SYNC();
        PSTAMP(PT_BAR_B);
        // ---------------------------------------------------------- phase R: row units (first unit of each warp: T2 load and
        // inverse x-FFT do not need the scalars, so they are issued before the scalar reduction)
        auto unit_stage1 = [&](const Unit &q) -> C2 * {     // T2 -> inverse x-FFT; returns the buffer holding the two rows
            const C2 *src = a.T2 + (((size_t)q.f * C + q.c) * npairs + q.j) * Ph * 2;
            C2 uu[5], vv[5];
#pragma unroll
            for (int m = 0; m < 5; ++m) { const int kk = lane + 32 * m; if (kk < Ph) ldcg_pair(src + 2 * kk, uu[m], vv[m]); }
#pragma unroll
            for (int m = 0; m < 5; ++m) {
                const int kk = lane + 32 * m;
                if (kk < Ph) {
                    bufA[kk] = mk<T>(uu[m].x - vv[m].y, uu[m].y + vv[m].x);                              // U_k + i V_k
                    if (kk > 0 && 2 * kk < P) bufA[P - kk] = mk<T>(uu[m].x + vv[m].y, vv[m].x - uu[m].y);   // conj(U_k) + i conj(V_k)
                }
            }
            return wfft<T, true>(bufA, bufB, *sfd, tw, lane);
        };
        auto unit_stage2 = [&](int i, const Unit &q, C2 *Z) {
            C2 *O = (Z == bufA) ? bufB : bufA;
            for (int e = lane; e < P; e += 32) O[e] = mk<T>((T)0, (T)0);
            __syncwarp();
            const double *sc = scal + q.f * SB;
            const T alpha = (T)sc[SC_ALPHA], beta = (T)sc[SC_BETA];
            const bool upd = sc[SC_UPD] != 0.0, step = sc[SC_ALPHA] != 0.0;
            const T c0 = (T)sc[SC_HEAD + 2 * C + q.w * 3 + q.comp], c2 = (T)sc[SC_HEAD + 2 * C + q.w * 3 + 2];
            T *ux = vec_x(i, q), *ur = vec_r(i, q), *up = vec_p(i, q);
            double rr = 0.0;
            for (int e = lane; e < q.len; e += 32) {
                const int ii = q.s0 + e;
                const bool row1 = ii >= q.s1;
                const int xc = s_ix[ii], y = row1 ? q.y0 + 1 : q.y0;
                const T coord = ((q.comp ? (T)y : (T)xc) - half_n) * dd;
                const T qp = (row1 ? Z[xc].y : Z[xc].x) - (c0 + c2 * coord);
                T rv;
                if (pre) {                                   // warm start: r = b - M_s q, p = r
                    rv = a.b[q.base + e] - qp;
                    ur[e] = rv; up[e] = rv;
                } else {
                    rv = ur[e];
                    T pv = up[e];
                    if (upd) { pv = rv + beta * pv; up[e] = pv; }
                    if (step) {
                        ux[e] += alpha * pv;
                        rv -= alpha * qp;
                        ur[e] = rv;
                    }
                }
                rr += (double)rv * (double)rv;
                if (row1) O[xc].y = rv; else O[xc].x = rv;
            }
            rr = warp_sum(rr);
            if (lane == 0) upart[i] = rr;
            fwd_rows_to_T1(O, Z, q);
        };
        Unit q0;
        C2 *Z0 = nullptr;
        const bool has0 = i_first < nu;
        if (has0) { q0 = unit_of(i_first); Z0 = unit_stage1(q0); }
        // scalars: alpha_k, mode coefficients
        for (int item = warp; item < F * NQ; item += NW) {
            const int f = item / NQ, qq = item - f * NQ;
            const double s = (qq == 0 || a.any_remove) ? warp_sum_cg160(a.part_s + ((size_t)f * NQ + qq) * Ph, Ph, lane) : 0.0;
            if (lane == 0) scal[f * SB + (qq == 0 ? SC_PQ : SC_HEAD + qq - 1)] = s;
        }
        __syncthreads();
        for (int t = tid; t < F * N; t += kPThreads) mode_coefs(t);
        if (!pre && tid >= 32 * (NW - 1) && tid - 32 * (NW - 1) < F) {       // last warp: alpha per frame (F <= 32 per pass)
            for (int f = tid - 32 * (NW - 1); f < F; f += 32) {
                double *sc = scal + f * SB;
                const double rho = sc[SC_RHO], pq = sc[SC_PQ];
                const double al = (rho > 0.0 && pq > 0.0) ? div_as<T>(rho, pq) : 0.0;     // breakdown: freeze (reading G16)
                sc[SC_ALPHA] = al;
                if (b == 0) a.alpha[f] = al;
            }
        }
        __syncthreads();
        PSTAMP(PT_SCAL);
        if (has0) unit_stage2(i_first, q0, Z0);
        for (int i = i_first + NW; i < nu; i += NW) {
            const Unit q = unit_of(i);
            C2 *Z = unit_stage1(q);
            unit_stage2(i, q, Z);
        }
        publish_rr();
        PSTAMP(PT_ROWS);
        GRID_SYNC();
        PSTAMP(PT_BAR_A);
    }
    k = -2;

    // ================================================================ tail: rho_{n_iter}; optional p = r + beta p; x, r, p -> global
    for (int f = warp; f < F; f += NW) {
        double rho;
        if (a.n_iter == 0 && a.mode == PM_STATE) rho = a.hist[(size_t)f * a.hist_stride];
        else rho = warp_sum_cg160(a.part_r + (size_t)f * G, G, lane);
        if (lane == 0) {
            double *sc = scal + f * SB;
            const double rho_prev = sc[SC_RHO];
            const bool upd = (a.n_iter > 0) && (sc[SC_ALPHA] != 0.0) && (rho_prev > 0.0);
            sc[SC_BETA] = upd ? div_as<T>(rho, rho_prev) : 0.0;
            sc[SC_UPD] = upd ? 1.0 : 0.0;
            if (b == 0) {
                a.hist[(size_t)f * a.hist_stride + a.n_iter] = rho;
                if (a.scal_out && f == 0) { a.scal_out[0] = rho; a.scal_out[1] = sc[SC_ALPHA]; a.scal_out[2] = sc[SC_BETA]; }
            }
        }
    }
    __syncthreads();
    for (int i = i_first; i < nu; i += NW) {
        const Unit q = unit_of(i);
        const double *sc = scal + q.f * SB;
        const bool fin = a.finalize_p && sc[SC_UPD] != 0.0;
        const T beta = (T)sc[SC_BETA];
        T *ux = vec_x(i, q), *ur = vec_r(i, q), *up = vec_p(i, q);
        if (!fin && !a.vec_smem) continue;
        for (int e = lane; e < q.len; e += 32) {
            T pv = up[e];
            const T rv = ur[e];
            if (fin) pv = rv + beta * pv;
            a.p[q.base + e] = pv;
            if (a.vec_smem) { a.x[q.base + e] = ux[e]; a.r[q.base + e] = rv; }
        }
    }
#undef PSTAMP
#undef GRID_SYNC
}

// ------------------------------------------------------------------------------------------------ host side
struct PersistState {
    unsigned *d_flags = nullptr;
    void *d_T1 = nullptr, *d_T1p = nullptr, *d_T2 = nullptr, *d_mspec = nullptr, *d_s2c = nullptr;
    double *d_part_r = nullptr, *d_part_s = nullptr, *d_part_i = nullptr;
    int G = 0, nq_m = 1, NQ = 0, SB = 0, any_remove = 0, spec_smem = 0, vec_smem = 0;
    int off_ms = 0, off_work = 0, off_scal = 0, off_wred = 0, off_tab = 0, off_upart = 0, off_rowptr = 0, off_ix = 0,
        off_vec = 0, off_spec = 0, wred_stride = 0;
    size_t smem = 0;
    bool attr_set = false;
};

#define PCK(call)                                                                 \
    do {                                                                          \
        cudaError_t e_ = (call);                                                  \
        if (e_ != cudaSuccess) {                                                  \
            set_error(std::string(#call) + ": " + cudaGetErrorString(e_));        \
            return TOMO_ECUDA;                                                    \
        }                                                                         \
    } while (0)

static int palloc(tomo_plan *pl, void **ptr, size_t bytes) {
    void *p = nullptr;
    bytes = std::max<size_t>(bytes, 16);
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) { set_error(std::string("cudaMalloc: ") + cudaGetErrorString(e)); return TOMO_ENOMEM; }
    pl->allocs.push_back(p);
    pl->bytes += bytes;
    *ptr = p;
    return TOMO_OK;
}

static size_t align16(size_t v) { return (v + 15) & ~(size_t)15; }

// spectra of the pupil mask and of the coordinate-weighted masks: [nq_m][Ph][P] complex fp64
static void build_mask_spectra(const HostModel &m, int nq_m, std::vector<std::complex<double>> &out) {
    const int P = m.P, Ph = m.Ph;
    out.assign((size_t)nq_m * Ph * P, 0.0);
    std::vector<std::complex<double>> img((size_t)P * P);
    for (int q = 0; q < nq_m; ++q) {
        std::fill(img.begin(), img.end(), 0.0);
        for (int i = 0; i < m.nv; ++i) {
            double wv = 1.0;
            if (q == 1) wv = (m.ix[i] - 0.5 * (m.n - 1)) * m.d;
            if (q == 2) wv = (m.iy[i] - 0.5 * (m.n - 1)) * m.d;
            img[(size_t)m.iy[i] * P + m.ix[i]] = wv;
        }
        for (int y = 0; y < P; ++y) host_fft(&img[(size_t)y * P], P, 1, false);      // along x
        for (int x = 0; x < P; ++x) host_fft(&img[x], P, P, false);                  // along y
        for (int kx = 0; kx < Ph; ++kx)
            for (int ky = 0; ky < P; ++ky) out[((size_t)q * Ph + kx) * P + ky] = img[(size_t)ky * P + kx];
    }
}

static int persist_prepare(tomo_plan *pl) {
    if (pl->persist) return TOMO_OK;
    const HostModel &m = pl->m;
    // Sigma_eta uniform per channel?
    for (int c = 0; c < m.C; ++c)
        for (int i = 1; i < m.nv; ++i)
            if (m.sigma2_full[(size_t)c * m.nv + i] != m.sigma2_full[(size_t)c * m.nv]) {
                set_error("persistent solver needs a noise variance that is uniform per WFS channel");
                return TOMO_EUNSUPPORTED;
            }
    int dev = 0, sms = 0, coop = 0, max_smem = 0;
    PCK(cudaGetDevice(&dev));
    PCK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    PCK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    PCK(cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    if (!coop) { set_error("device does not support cooperative launches"); return TOMO_EUNSUPPORTED; }
    if (m.Ph > sms || m.Ph > 160 || sms > 160) { set_error("persistent solver: more k_x slabs than SMs (or than 160)"); return TOMO_EUNSUPPORTED; }
    if ((m.P + 31) / 32 > kPWarps) { set_error("persistent solver: FFT edge too large"); return TOMO_EUNSUPPORTED; }
    if (m.nv >= 65536 || m.C * ((m.n + 1) / 2) > 2 * kPThreads) { set_error("persistent solver: grid too large"); return TOMO_EUNSUPPORTED; }
    PersistState *ps = new PersistState();
    const int npairs = (m.n + 1) / 2, U = m.C * npairs, F = pl->F;
    ps->G = std::max(1, std::min(sms, std::max(F * U, m.Ph)));
    ps->any_remove = 0;
    bool focus = false;
    for (int i = 0; i < m.n_wfs; ++i) { if (m.n_remove[i] > 0) ps->any_remove = 1; if (m.n_remove[i] > 2) focus = true; }
    ps->nq_m = focus ? 3 : 1;
    ps->NQ = 1 + m.C * (focus ? 2 : 1);
    ps->SB = SC_HEAD + 2 * m.C + 3 * m.n_wfs;
    const size_t E = pl->elem, SE = pl->selem;
    const int WPG = (m.P + 31) / 32, Goc = std::min(kPWarps / WPG, m.C), OCG = (m.C + Goc - 1) / Goc;
    const int maxu = (F * U + ps->G - 1) / ps->G;
    ps->wred_stride = 1 + 2 * OCG;
    size_t off = (size_t)m.P * 2 * E;
    ps->off_ms = (int)(off = align16(off));
    off += (size_t)ps->nq_m * m.P * 2 * E;
    ps->off_work = (int)(off = align16(off));
    off += (size_t)std::max(2 * m.C, 2 * kPWarps) * m.P * 2 * E;
    ps->off_scal = (int)(off = align16(off));
    off += (size_t)F * ps->SB * sizeof(double);
    ps->off_wred = (int)(off = align16(off));
    off += (size_t)kPWarps * ps->wred_stride * sizeof(double);
    ps->off_tab = (int)(off = align16(off));
    off += (size_t)m.n_wfs * (9 * sizeof(double) + sizeof(int)) + 8 + (size_t)(m.C + 2) * E + sizeof(FftDesc) + 16;
    ps->off_upart = (int)(off = align16(off));
    off += (size_t)maxu * sizeof(double);
    ps->off_rowptr = (int)(off = align16(off));
    off += (size_t)(m.n + 1) * sizeof(int);
    ps->off_ix = (int)(off = align16(off));
    off += (size_t)m.nv * sizeof(unsigned short);
    off = align16(off);
    const size_t spec_bytes = (size_t)m.n_pair * m.P * 2 * SE, vec_bytes = (size_t)maxu * 6 * m.n * E;
    const char *no_pin = getenv("TOMO_NO_SPEC_SMEM"), *no_vec = getenv("TOMO_NO_VEC_SMEM");
    // the spectra slice has priority for the shared memory that is left, then the CG vectors of the CTA's row units
    ps->off_spec = (int)off;
    ps->spec_smem = (off + spec_bytes <= (size_t)max_smem) && !(no_pin && no_pin[0] == '1');
    if (ps->spec_smem) off = align16(off + spec_bytes);
    ps->off_vec = (int)off;
    ps->vec_smem = (off + vec_bytes <= (size_t)max_smem) && !(no_vec && no_vec[0] == '1');
    if (ps->vec_smem) off = align16(off + vec_bytes);
    if (off > (size_t)max_smem) { delete ps; set_error("persistent solver: problem too large for shared memory"); return TOMO_EUNSUPPORTED; }
    ps->smem = off;

    int rc;
#define PTRY(x) do { rc = (x); if (rc) { delete ps; return rc; } } while (0)
    const size_t tsz = (size_t)F * m.Ph * m.C * 2 * npairs * 2 * E;
    PTRY(palloc(pl, (void **)&ps->d_flags, 1024));
    PTRY(palloc(pl, &ps->d_T1, tsz));
    PTRY(palloc(pl, &ps->d_T1p, tsz));
    PTRY(palloc(pl, &ps->d_T2, tsz));
    PTRY(palloc(pl, (void **)&ps->d_part_r, (size_t)F * sms * sizeof(double)));
    PTRY(palloc(pl, (void **)&ps->d_part_s, (size_t)F * m.Ph * ps->NQ * sizeof(double)));
    PTRY(palloc(pl, (void **)&ps->d_part_i, (size_t)F * U * 2 * sizeof(double)));
    PTRY(palloc(pl, &ps->d_mspec, (size_t)ps->nq_m * m.Ph * m.P * 2 * E));
    PTRY(palloc(pl, &ps->d_s2c, (size_t)m.C * E));
#undef PTRY
    std::vector<std::complex<double>> msp;
    build_mask_spectra(m, ps->nq_m, msp);
    std::vector<double> s2(m.C);
    for (int c = 0; c < m.C; ++c) s2[c] = m.sigma2_full[(size_t)c * m.nv] / ((double)m.P * m.P);
    if (E == 8) {
        PCK(cudaMemcpy(ps->d_mspec, msp.data(), msp.size() * 16, cudaMemcpyHostToDevice));
        PCK(cudaMemcpy(ps->d_s2c, s2.data(), s2.size() * 8, cudaMemcpyHostToDevice));
    } else {
        std::vector<float> mf(msp.size() * 2), sf(s2.begin(), s2.end());
        for (size_t i = 0; i < msp.size(); ++i) { mf[2 * i] = (float)msp[i].real(); mf[2 * i + 1] = (float)msp[i].imag(); }
        PCK(cudaMemcpy(ps->d_mspec, mf.data(), mf.size() * 4, cudaMemcpyHostToDevice));
        PCK(cudaMemcpy(ps->d_s2c, sf.data(), sf.size() * 4, cudaMemcpyHostToDevice));
    }
    pl->persist = ps;
    return TOMO_OK;
}

template <typename T, typename S>
static int persist_launch(tomo_plan *pl, cudaStream_t st, int F, int n_iter, int mode, int finalize_p, const float *slopes,
                          const float *x0, double *scal_out, long long *dbg = nullptr) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    PersistState *ps = (PersistState *)pl->persist;
    const HostModel &m = pl->m;
    PArgs<T, S> a;
    std::memset(&a, 0, sizeof(a));
    a.st.fd = pl->fd; a.st.P = m.P; a.st.Ph = m.Ph; a.st.tw = (const C2 *)pl->d_tw;
    a.g = pl->g;
    a.F = F; a.n_iter = n_iter; a.mode = mode; a.finalize_p = finalize_p;
    a.npad = 2 * pl->g.npairs; a.U = m.C * pl->g.npairs; a.NQ = ps->NQ; a.nq_m = ps->nq_m; a.SB = ps->SB;
    a.G = std::max(1, std::min(ps->G, std::max(F * a.U, m.Ph)));
    a.spec_smem = ps->spec_smem; a.any_remove = ps->any_remove;
    a.off_ms = ps->off_ms; a.off_work = ps->off_work; a.off_scal = ps->off_scal; a.off_wred = ps->off_wred;
    a.off_tab = ps->off_tab; a.off_upart = ps->off_upart; a.off_rowptr = ps->off_rowptr; a.off_ix = ps->off_ix;
    a.off_vec = ps->off_vec; a.off_spec = ps->off_spec; a.wred_stride = ps->wred_stride; a.vec_smem = ps->vec_smem;
    a.s_in = slopes; a.x0 = x0;
    a.x = (T *)pl->d_x; a.r = (T *)pl->d_r; a.p = (T *)pl->d_p; a.b = (T *)pl->d_b;
    a.T1 = (C2 *)ps->d_T1; a.T1p = (C2 *)ps->d_T1p; a.T2 = (C2 *)ps->d_T2;
    a.spec = (const S2 *)pl->d_spec; a.n_pair = m.n_pair;
    a.mspec = (const C2 *)ps->d_mspec; a.s2c = (const T *)ps->d_s2c;
    a.part_r = ps->d_part_r; a.part_s = ps->d_part_s; a.part_i = ps->d_part_i;
    a.hist = pl->d_hist; a.hist_stride = pl->hist_cap; a.alpha = pl->d_alpha; a.scal_out = scal_out;
    a.flags = ps->d_flags; a.dbg = dbg;
    if (!ps->attr_set) {
        PCK(cudaFuncSetAttribute((k_persistent<T, S>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ps->smem));
        int occ = 0;
        PCK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (k_persistent<T, S>), kPThreads, ps->smem));
        if (occ < 1) { set_error("persistent kernel does not fit on an SM"); return TOMO_EUNSUPPORTED; }
        ps->attr_set = true;
    }
    PCK(cudaMemsetAsync(ps->d_flags, 0, 1024, st));
    void *kargs[] = {&a};
    PCK(cudaLaunchCooperativeKernel((const void *)(k_persistent<T, S>), dim3(a.G), dim3(kPThreads), kargs, ps->smem, st));
    pl->launches_last += 1;
    return TOMO_OK;
}

static int persist_dispatch(tomo_plan *pl, cudaStream_t st, int F, int n_iter, int mode, int finalize_p, const float *slopes,
                            const float *x0, double *scal_out, long long *dbg = nullptr) {
    if (pl->opt.precision == TOMO_F32) return persist_launch<float, float>(pl, st, F, n_iter, mode, finalize_p, slopes, x0, scal_out, dbg);
    if (pl->opt.precision == TOMO_F32S_F64A) return persist_launch<double, float>(pl, st, F, n_iter, mode, finalize_p, slopes, x0, scal_out, dbg);
    return persist_launch<double, double>(pl, st, F, n_iter, mode, finalize_p, slopes, x0, scal_out, dbg);
}

int project_from_x(tomo_plan *pl, cudaStream_t st, int F);       // tomo_api.cu: A7-A8 from d_x -> d_out
int state_load(tomo_plan *pl, cudaStream_t st, const float *x, const float *r, const float *p, const double *rho);
int state_store(tomo_plan *pl, cudaStream_t st, float *x, float *r, float *p);

int solve_persistent(tomo_plan *pl, const float *slopes, float *out, int F, int n_iter, const float *x0, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    pl->launches_last = 0;
    if ((rc = persist_dispatch(pl, st, F, n_iter, x0 ? PM_WARM : PM_COLD, 0, slopes, x0, nullptr))) return rc;
    if (pl->has_cos && out) {
        if ((rc = project_from_x(pl, st, F))) return rc;
        PCK(cudaMemcpyAsync(out, pl->d_out, (size_t)F * pl->m.T * pl->m.nvp * sizeof(float), cudaMemcpyDeviceToDevice, st));
    }
    pl->last_frames = F; pl->last_iter = n_iter;
    return TOMO_OK;
}

// one teacher-forced iteration through the persistent kernel (tomo_cg_step with the persistent solver)
int cg_step_persistent(tomo_plan *pl, float *x, float *r, float *p, double *scal, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    pl->launches_last = 0;
    if ((rc = state_load(pl, st, x, r, p, scal))) return rc;
    if ((rc = persist_dispatch(pl, st, 1, 1, PM_STATE, 1, nullptr, nullptr, scal))) return rc;
    return state_store(pl, st, x, r, p);
}

// Measurement aid (tomo_time_phases): one instrumented persistent solve from the state the last solve left
// (PM_STATE), thread 0 of every CTA stamps clock64 at the phase boundaries; returns, per segment, the mean over
// iterations of the MAXIMUM over CTAs (work segments) or the MINIMUM over CTAs (barrier waits = pure latency).
int time_phases_persistent(tomo_plan *pl, int F, int n_iter, float *us_out, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    PersistState *ps = (PersistState *)pl->persist;
    const int G = std::max(1, std::min(ps->G, std::max(F * pl->m.C * pl->g.npairs, pl->m.Ph)));
    long long *d_dbg = nullptr;
    const size_t cnt = (size_t)G * n_iter * PT_N;
    PCK(cudaMalloc(&d_dbg, cnt * sizeof(long long)));
    PCK(cudaMemsetAsync(d_dbg, 0, cnt * sizeof(long long), st));
    rc = persist_dispatch(pl, st, F, n_iter, PM_STATE, 0, nullptr, nullptr, nullptr, d_dbg);
    std::vector<long long> h(cnt);
    cudaError_t e = cudaStreamSynchronize(st);
    if (!rc && e == cudaSuccess) e = cudaMemcpy(h.data(), d_dbg, cnt * sizeof(long long), cudaMemcpyDeviceToHost);
    cudaFree(d_dbg);
    if (rc) return rc;
    if (e != cudaSuccess) { set_error(std::string("time_phases: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, pl->device);
    const double us_per_cycle = 1e3 / std::max(khz, 1);
    for (int s = 0; s < PT_N; ++s) us_out[s] = 0.f;
    for (int k = 0; k < n_iter; ++k)
        for (int s = 1; s < PT_N; ++s) {
            const bool wait = (s == PT_BAR_B || s == PT_BAR_A);
            const bool slab_seg = (s >= PT_BUILD && s <= PT_INV);
            long long best = wait ? (1LL << 62) : 0;
            for (int b = 0; b < G; ++b) {
                const long long *t = &h[((size_t)b * n_iter + k) * PT_N];
                const bool has_slab = t[PT_MAC] != 0;
                if (slab_seg && !has_slab) continue;
                if (s == PT_BAR_B && !has_slab) continue;
                const long long prev = (s == PT_BAR_B && !has_slab) ? t[PT_RHO] : t[s - 1];
                const long long dt = t[s] - prev;
                best = wait ? std::min(best, dt) : std::max(best, dt);
            }
            us_out[s] += (float)(best * us_per_cycle / n_iter);
        }
    // total per iteration as seen by CTA 0
    us_out[0] = n_iter > 1 ? (float)((h[((size_t)(n_iter - 1)) * PT_N + PT_BAR_A] - h[PT_START]) * us_per_cycle / n_iter) : 0.f;
    return TOMO_OK;
}

void persist_destroy(tomo_plan *pl) {
    delete (PersistState *)pl->persist;
    pl->persist = nullptr;
}

}  // namespace tomo
