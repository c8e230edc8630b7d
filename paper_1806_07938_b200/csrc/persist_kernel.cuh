// persist_kernel.cuh -- persistent cooperative CG solver: ONE kernel per solve, two grid barriers per iteration,
// every 1-D transform held in registers (fft_reg.cuh: two passes, one shared-memory exchange).
//
// The textbook CG recurrences (PAPER.md S2.G L337, Eq.12) are kept, but the work is re-ordered so that an
// iteration has only the two all-to-all exchanges the 2-D FFT itself needs:
//
//   phase C_k (one CTA per k_x slab, all channels):   rho_k, beta_k from the r.r partials;
//        p~rows_k = r~rows_k + beta_k p~rows_{k-1}    (the x-FFT is linear, so p = r + beta p is formed in the
//                                                      half-transformed domain; p~rows stays with its slab)
//        y-FFT, per-frequency C x C block product with the Hermitian-packed kernel spectra pinned in shared
//        memory (Eq.22, Eq.30), + sigma^2 p~ (Sigma_eta, L260), inverse y-FFT -> T2
//        p.q and the modal sums Z^T q (Eq.36) by Parseval from p~, y~ and the mask spectra
//   ---- grid barrier B ----
//   phase R_k (16 lanes per (channel, row pair)):      alpha_k = rho_k / p.q, mode coefficients;
//        inverse x-FFT, crop + mask (S_2, W_s; Eq.24-27, Eq.34), q' = M_s q,
//        p_k = r_k + beta_k p_{k-1} (spatial copy), x += alpha p, r -= alpha q', partial r.r,
//        forward x-FFT of the NEW residual rows (S_1, Eq.18-21) -> T1
//   ---- grid barrier A ----
//
// p.q is taken in the frequency domain (Parseval; p is zero outside the pupil, so the crop does not matter and
// p.M_s q = p.q for p in range(M_s)); every reduction is a fixed-order sum with fp64 scalars, so a fixed-count
// solve is bit-reproducible.  Sigma_eta must be uniform per channel here (all configs).
//
// Every 1-D transform is the same two shared-memory-to-shared-memory passes (P = A * B, A <= B <= 16; fft_reg.cuh):
//   pass 1  thread j2 < B:  radix A over j = j1 B + j2, twiddle W_P^{j2 k1}  -> Y[k1 (B+1) + j2]
//   pass 2  thread k1 < A:  radix B over j2                                  -> X[k1 + A k2]
// done by TWO small non-inlined codelets that the slab phase, the row phase, the forward and the inverse transforms
// all share (an inverse transform is the forward one on conjugated data: conj on the way in, conj on the way out).
// The whole per-iteration instruction footprint has to stay within the 32 KB L1.5 instruction cache: the first
// register-FFT version of this kernel was fully unrolled (333 KB of SASS) and stalled on instruction fetch.
#pragma once
#include <cuda_runtime.h>

#include "fft_reg.cuh"
#include "tomo_kernels.cuh"

namespace tomo {

static const int kPThreads = 512;
static const int kPWarps = kPThreads / 32;
static const int kGS = 16;                       // lanes per row unit

enum { PM_COLD = 0, PM_WARM = 1, PM_STATE = 2, PM_APPLY = 3 };   // PM_APPLY: one product, r <- M_s A M_s v (tomo_apply_css)
enum { PT_START = 0, PT_RHO = 1, PT_BUILD = 2, PT_FFT = 3, PT_MAC = 4, PT_INV = 5, PT_BAR_B = 6, PT_SCAL = 7, PT_ROWS = 8, PT_BAR_A = 9, PT_R_LOAD = 10, PT_R_FFT1 = 11, PT_R_UPD = 12, PT_R_FFT2 = 13, PT_N = 16 };

// per-frame scalar block in shared memory (doubles)
enum { SC_RHO = 0, SC_RHO_PREV = 1, SC_BETA = 2, SC_ALPHA = 3, SC_UPD = 4, SC_PQ = 5, SC_HEAD = 6 };
// ... followed by the 2C channel sums of q, the 3N mode coefficients, and (MINRES) the 2C channel sums of v_k and the state of
// the Paige-Saunders recurrences at offset SC_HEAD + 4C + 3N:
enum { MR_C = 0, MR_S = 1, MR_DBAR = 2, MR_EPS = 3, MR_PHIBAR = 4, MR_FROZEN = 5, MR_BETA = 6, MR_INVBETA = 7,
       MR_PON = 8, MR_PEPS = 9, MR_PDELTA = 10, MR_PINVG = 11, MR_PPHI = 12, MR_N = 16 };
enum { METHOD_CG = 0, METHOD_MINRES = 1 };

template <typename T, typename S> struct PArgs {
    DevGeom g;
    int P, Ph;
    const typename cx_of<T>::type *tw;   // device [P], exp(-2 pi i t/P)
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
    int off_ms, off_work, off_red, off_scal, off_tab, off_upart, off_vm, off_vec, off_spec, off_ptab, off_unit;
    int ngs;                     // row-unit buffer slots in shared memory = row units processed per round
    int off_ms2;                 // mask spectra of the helped slab
    int fb;                      // batch instance: frames per slab pass (1 or 2: two frames share the four FFT passes)
    const int *seg;              // [G][8] slab work of a CTA: own frames [0],[1]; helped slab k_x [2], frames [3],[4] (balance)
    const float *s_in;           // [F][C][nv] slopes (COLD/WARM)
    const float *x0;             // [F][C][nv] warm start (WARM)
    T *x, *r, *p;                // [F][C][nv] valid-only layout (ABI side)
    T *xd, *rd, *pd, *bd;        // [F][C][npad][n] dense rows (solver side; xd/rd/pd unused with vec_smem)
    T *w1d, *w2d;                // MINRES: dense rows of w_{k-1}, w_{k-2} (unused with vec_smem)
    typename cx_of<T>::type *T1;    // [F][Ph][C][npad]     x-FFT of the current residual rows
    typename cx_of<T>::type *T1p;   // [F][Ph][C][npad]     x-FFT of the search direction (slab-private state)
    typename cx_of<T>::type *T2;    // [F][C][npairs][Ph][2]
    const typename cx_of<S>::type *spec;   // [Ph][n_pair][P]
    int n_pair;
    const typename cx_of<T>::type *mspec;  // [nq_m][Ph][P]  spectra of the pupil mask (and coordinate-weighted masks)
    const T *s2c;                // [C] sigma^2_c / P^2
    double *part_r;              // [F][U]       r.r per row unit
    double *part_s;              // [F][NQ][Ph]  per slab: p.q, sum q_c, sum coord q_c
    double *part_i;              // [F][U][2]    init: sum s, sum coord s per row unit
    double *hist;                // [F][hist_stride] rho_k
    int hist_stride;
    double *alpha;               // [F]
    double *scal_out;            // [3] rho_{k+1}, alpha, beta (finalize_p, frame 0) or NULL
    unsigned *flags;             // arrival counter of the grid barrier
    long long *dbg;              // [G][n_iter][PT_N] clock64 stamps of thread 0 (measurement aid) or NULL
};

// ---- grid barrier: one arrival counter.  Writers: data stores -> bar.sync -> thread 0: red.release.
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

// sum over the 16 lanes of a row-unit group (every lane of the group returns the total)
__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
    for (int o = kGS / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Modal sums against G = (Z^T Z)^-1 of one WFS (3 x 3, rows / columns beyond n_remove are zero; Eq.36).  The loops run
// to the constant 3 under a predicate so that the three-element arrays stay in registers: a loop to n_remove indexes them
// dynamically and sends them to local memory (measured: 3 us per MINRES iteration at cfg3).
__device__ __forceinline__ double modal_quad(const double *G, const double tp[3], const double tq[3], int nr) {
    double t = 0.0;
#pragma unroll
    for (int u = 0; u < 3; ++u) {
        double sq = 0.0;
#pragma unroll
        for (int v = 0; v < 3; ++v) if (v < nr) sq += G[u * 3 + v] * tq[v];
        if (u < nr) t += tp[u] * sq;
    }
    return t;
}
__device__ __forceinline__ void modal_coef(const double *G, const double tq[3], int nr, int comp, double &d0, double &d2) {
    d0 = 0.0; d2 = 0.0;
#pragma unroll
    for (int v = 0; v < 3; ++v) if (v < nr) { d0 += G[comp * 3 + v] * tq[v]; d2 += G[6 + v] * tq[v]; }
}

// deterministic sum by one warp of up to 160 contiguous doubles other CTAs wrote: all loads in flight at once
__device__ __forceinline__ double warp_sum_cg160(const double *src, int count, int lane) {
    double v[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) { const int i = lane + 32 * m; v[m] = (i < count) ? __ldcg(src + i) : 0.0; }
    return warp_sum(((v[0] + v[1]) + (v[2] + v[3])) + v[4]);
}
// fixed-order sum by one warp of `count` contiguous doubles other CTAs wrote, 16 loads in flight per lane
__device__ __forceinline__ double warp_sum_units(const double *src, int count, int lane) {
    double acc = 0.0;
    for (int i0 = 0; i0 < count; i0 += 512) {
        double v[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) { const int i = i0 + m * 32 + lane; v[m] = __ldcg(src + min(i, count - 1)); if (i >= count) v[m] = 0.0; }
#pragma unroll
        for (int m = 8; m > 0; m >>= 1)
#pragma unroll
            for (int j = 0; j < m; ++j) v[j] += v[j + m];
        acc += v[0];
    }
    return warp_sum(acc);
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
__device__ __forceinline__ void st_pair(float2 *p, float2 u, float2 v) { *reinterpret_cast<float4 *>(p) = make_float4(u.x, u.y, v.x, v.y); }
__device__ __forceinline__ void st_pair(double2 *p, double2 u, double2 v) { p[0] = u; p[1] = v; }
__device__ __forceinline__ float2 shfl_c(float2 v, int src) {
    return make_float2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}
__device__ __forceinline__ double2 shfl_c(double2 v, int src) {
    return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}

// ---- the two codelets: R-point DFT from src (stride ss; only the first nin inputs are read, the rest are zero: the
// padding of Eq.18-19 is never stored) to dst (stride ds), optional twiddle tw[tj * k]
template <typename T, int R, bool TW>
__device__ __noinline__ void dft_pass(const typename cx_of<T>::type *src, int ss, int nin, typename cx_of<T>::type *dst, int ds,
                                      const typename cx_of<T>::type *tw, int tj) {
    typedef typename cx_of<T>::type C2;
    C2 v[R], w[TW ? R : 1];
#pragma unroll
    for (int j = 0; j < R; ++j) v[j] = (j < nin) ? src[j * ss] : mk<T>((T)0, (T)0);
    // the twiddles go into registers beside the data: loaded one by one between the stores below (which may alias the
    // table as far as the compiler knows) they put R - 1 shared-memory round trips into the pass (measured on the B200, one
    // warp, radix 10 of P = 160: 609 -> 400 cycles per pass)
    if (TW) {
#pragma unroll
        for (int k = 1; k < R; ++k) w[k] = tw[tj * k];
    }
    SmallDft<T, R, false>::run(v);
    dst[0] = v[0];
#pragma unroll
    for (int k = 1; k < R; ++k) dst[k * ds] = TW ? cmul(v[k], w[k]) : v[k];
}

struct PairRef { int off; float sgn; };
struct UnitRec { int f, c, j, s0, s1, s2, pad0, pad1; };   // row unit of a CTA: frame, channel, row pair, valid-list range          // spectrum block of (c_out, c_in): element offset and conjugation sign

// ---- the rows [LO, HI) of the block product for one k_y, straight-line: every pair index and conjugation is a
// compile-time constant, no branch between the rows (the loads of the next row overlap the FMAs of this one)
template <typename T, typename S, int CT, int PP, int LO, int HI, bool MR = false>
__device__ __forceinline__ void mac_rows(const typename cx_of<T>::type (&x)[CT], const typename cx_of<S>::type *sp, const T *s2c,
                                         typename cx_of<T>::type *Y, int LD, int ky, typename cx_of<T>::type m0,
                                         typename cx_of<T>::type m1, typename cx_of<T>::type m2, T *red_s, T *red_f,
                                         int any_remove, int nq_m, T &pap) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    // input channel outermost: the HI - LO outputs of the group advance together (2 (HI - LO) independent accumulator chains);
    // the terms of an output still arrive in the order c_in = 0 .. C-1
    T ar[HI - LO], ai[HI - LO];
#pragma unroll
    for (int o = 0; o < HI - LO; ++o) { const T s2 = s2c[LO + o]; ar[o] = s2 * x[LO + o].x; ai[o] = s2 * x[LO + o].y; }
#pragma unroll
    for (int ci = 0; ci < CT; ++ci) {
#pragma unroll
        for (int o = 0; o < HI - LO; ++o) {
            const int oc = LO + o;
            const int lo = ci < oc ? ci : oc, hi = ci < oc ? oc : ci;
            const S2 s = sp[(lo * CT - (lo * (lo - 1)) / 2 + hi - lo) * PP];
            const T sr = (T)s.x, si = (T)s.y;
            if (ci < oc) {           // conjugate of the stored block
                ar[o] = fma(sr, x[ci].x, ar[o]); ar[o] = fma(si, x[ci].y, ar[o]);
                ai[o] = fma(sr, x[ci].y, ai[o]); ai[o] = fma(-si, x[ci].x, ai[o]);
            } else {
                ar[o] = fma(sr, x[ci].x, ar[o]); ar[o] = fma(-si, x[ci].y, ar[o]);
                ai[o] = fma(sr, x[ci].y, ai[o]); ai[o] = fma(si, x[ci].x, ai[o]);
            }
        }
    }
#pragma unroll
    for (int o = 0; o < HI - LO; ++o) {
        const int oc = LO + o;
        Y[oc * LD + ky] = mk<T>(ar[o], -ai[o]);
        pap += x[oc].x * ar[o] + x[oc].y * ai[o];                       // Re(conj(p~) y~)
        if (any_remove) {
            red_s[oc * PP + ky] = m0.x * ar[o] + m0.y * ai[o];          // Re(conj(m~) y~)
            if (nq_m > 1) { const C2 mm = (oc & 1) ? m2 : m1; red_f[oc * PP + ky] = mm.x * ar[o] + mm.y * ai[o]; }
            if (MR) {
                T *red_v = red_s + (nq_m > 1 ? 2 : 1) * CT * PP;
                const T ip2 = (T)1 / ((T)PP * (T)PP);
                red_v[oc * PP + ky] = ip2 * (m0.x * x[oc].x + m0.y * x[oc].y);
                if (nq_m > 1) { const C2 mm = (oc & 1) ? m2 : m1; red_v[(CT + oc) * PP + ky] = ip2 * (mm.x * x[oc].x + mm.y * x[oc].y); }
            }
        }
    }
}
template <typename T, typename S, int CT, int PP, int G, bool MR = false>
__device__ __forceinline__ void mac_dispatch(int grp, const typename cx_of<T>::type (&x)[CT], const typename cx_of<S>::type *sp,
                                             const T *s2c, typename cx_of<T>::type *Y, int LD, int ky, typename cx_of<T>::type m0,
                                             typename cx_of<T>::type m1, typename cx_of<T>::type m2, T *red_s, T *red_f,
                                             int any_remove, int nq_m, T &pap) {
    constexpr int WPG = (PP + 31) / 32, GOC = (kPWarps / WPG) < CT ? (kPWarps / WPG) : CT;
    if (grp == G) mac_rows<T, S, CT, PP, G * CT / GOC, (G + 1) * CT / GOC, MR>(x, sp, s2c, Y, LD, ky, m0, m1, m2, red_s, red_f, any_remove, nq_m, pap);
    else if constexpr (G + 1 < GOC) mac_dispatch<T, S, CT, PP, G + 1, MR>(grp, x, sp, s2c, Y, LD, ky, m0, m1, m2, red_s, red_f, any_remove, nq_m, pap);
}

// ---- per-frequency block product of one k_x slab (Eq.22, Eq.30) + Sigma_eta (L260) + Parseval partials.
// Warps are grouped: WPG = ceil(P/32) warps cover the k_y range, group g owns a contiguous range of output channels.
// X: forward y-spectra [c][LD] in natural k_y order; Y: [c][LD], CONJUGATED (the inverse transform is run as a forward
// one).  CT > 0: the C inputs of this k_y are held in registers; CT = 0: run-time channel count.
// red: [Goc][P] partial p.q, then [C][P] mask sums, then [C][P] focus sums.
template <typename T, typename S, int CT, int PP, bool MR>
__device__ __forceinline__ void mac_slab(const typename cx_of<T>::type *X, typename cx_of<T>::type *Y, int LD,
                                         const typename cx_of<S>::type *spec, const PairRef *ptab,
                                         const typename cx_of<T>::type *ms, const T *s2c,
                                         int C, int P, int nq_m, int any_remove, T *red, int warp, int lane) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    const int WPG = (P + 31) >> 5;
    const int Goc = min(kPWarps / WPG, C);
    const int grp = warp / WPG, ky = (warp - grp * WPG) * 32 + lane;
    if (grp >= Goc || ky >= P) return;
    const int oc_lo = grp * C / Goc, oc_hi = (grp + 1) * C / Goc;
    C2 m0 = mk<T>((T)0, (T)0), m1 = m0, m2 = m0;
    if (any_remove) { m0 = ms[ky]; if (nq_m > 1) { m1 = ms[P + ky]; m2 = ms[2 * P + ky]; } }
    T *red_s = red + Goc * P, *red_f = red_s + C * P;
    const S2 *sp = spec + ky;
    C2 x[CT > 0 ? CT : 1];
    if (CT > 0) {
#pragma unroll
        for (int ci = 0; ci < CT; ++ci) x[ci] = X[ci * LD + ky];
    }
    T pap = (T)0;
    if constexpr (CT > 0) {
        mac_dispatch<T, S, CT, PP, 0, MR>(grp, x, sp, s2c, Y, LD, ky, m0, m1, m2, red_s, red_f, any_remove, nq_m, pap);
    } else {
#pragma unroll 1
        for (int oc = oc_lo; oc < oc_hi; ++oc) {
            const C2 xo = X[oc * LD + ky];
            const T s2 = s2c[oc];
            const PairRef *row = ptab + oc * C;
            T ar = s2 * xo.x, ai = s2 * xo.y;
            for (int ci = 0; ci < C; ++ci) {
                const PairRef e = row[ci];
                const S2 s = sp[e.off];
                const C2 xv = X[ci * LD + ky];
                const T sr = (T)s.x, si = (T)s.y * (T)e.sgn;
                ar = fma(sr, xv.x, ar); ar = fma(-si, xv.y, ar);
                ai = fma(sr, xv.y, ai); ai = fma(si, xv.x, ai);
            }
            Y[oc * LD + ky] = mk<T>(ar, -ai);
            pap += xo.x * ar + xo.y * ai;
            if (any_remove) {
                red_s[oc * P + ky] = m0.x * ar + m0.y * ai;
                if (nq_m > 1) { const C2 mm = (oc & 1) ? m2 : m1; red_f[oc * P + ky] = mm.x * ar + mm.y * ai; }
            }
        }
    }
    red[grp * P + ky] = pap;
    if (MR && any_remove && CT == 0) {        // MINRES: the same modal sums of the product's INPUT v~ (every v_k is re-projected, reading G27; CT > 0: in mac_rows)
        T *red_v = red_s + (nq_m > 1 ? 2 : 1) * C * P;
        const T ip2 = (T)1 / ((T)P * (T)P);           // v~ is an unnormalised transform (y~ carries the 1/P^2 folded into the kernel spectra)
        for (int oc = oc_lo; oc < oc_hi; ++oc) {
            const C2 xo = X[oc * LD + ky];
            red_v[oc * P + ky] = ip2 * (m0.x * xo.x + m0.y * xo.y);
            if (nq_m > 1) { const C2 mm = (oc & 1) ? m2 : m1; red_v[(C + oc) * P + ky] = ip2 * (mm.x * xo.x + mm.y * xo.y); }
        }
    }
}

// fixed-order sum of `cnt` values of the slab partial array by one warp
template <typename T> __device__ __forceinline__ double warp_sum_red(const T *src, int cnt, int lane) {
    T s = (T)0;
    for (int i0 = 0; i0 < cnt; i0 += 256) {          // eight loads in flight, added in the order i = lane, lane + 32, ...
        T v[8];
#pragma unroll
        for (int m = 0; m < 8; ++m) { const int i = i0 + lane + 32 * m; v[m] = i < cnt ? src[i] : (T)0; }
#pragma unroll
        for (int m = 0; m < 8; ++m) s += v[m];
    }
    return warp_sum((double)s);
}

// BATCH = false: the single-frame instance (latency-bound: compact code, the CTA's own slab only);
// BATCH = true: several frames per solve (throughput: balanced slab passes, every global load of a step issued up front).
// PROF = true: thread 0 stamps clock64 at the phase boundaries (tomo_time_phases); the production instances carry no stamp code.
// METHOD_MINRES: the Paige-Saunders recurrences (the solver the paper keeps for the Toeplitz method, S2.G L337, L426; written
// out in oracle/solver.py:minres, reading G27) in the SAME two phases: the product's input is v_k = u_{k-1} / beta_k (the row
// phase sends the transform of the unnormalised u, phase C scales it: the transform is linear), alpha_k = v_k . M_s A v_k by
// Parseval where CG takes p.q, beta_{k+1} = |u_k| where CG takes r.r; the Givens rotation k needs beta_{k+1}, so x_k and w_k are
// updated one row phase later (the last one in the tail).  Rows of a unit: x, v_{k-1} (CG's r), u_{k-1} (CG's p), w_{k-1}, w_{k-2}.
template <typename T, typename S, int P, bool BATCH, bool PROF, int METHOD = METHOD_CG>
__global__ void __launch_bounds__(kPThreads, 1) k_persistent(PArgs<T, S> a) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    constexpr int A = Fact2<P>::A, B = Fact2<P>::B, Ph = P / 2 + 1;
    constexpr int LD = A * (B + 1);               // row stride of the slab buffers and size of a pass-1 result
    static_assert(A * B == P && A >= 2 && A <= B && B <= kGS, "unsupported split");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = a.g.n, nv = a.g.nv, C = a.g.C, npairs = a.g.npairs, N = a.g.N;
    const int F = a.F, U = a.U, NQ = a.NQ, SB = a.SB, G = a.G, npad = a.npad;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, NW = kPWarps, b = blockIdx.x;
    const int gl = lane & (kGS - 1), gs = tid / kGS;      // lane within the row-unit group, group slot
    C2 *tw = reinterpret_cast<C2 *>(smem_raw);
    C2 *ms = reinterpret_cast<C2 *>(smem_raw + a.off_ms);
    C2 *ms2 = reinterpret_cast<C2 *>(smem_raw + a.off_ms2);
    C2 *work = reinterpret_cast<C2 *>(smem_raw + a.off_work);
    T *red = reinterpret_cast<T *>(smem_raw + a.off_red);
    double *scal = reinterpret_cast<double *>(smem_raw + a.off_scal);
    double *sGs = reinterpret_cast<double *>(smem_raw + a.off_tab);
    int *s_nrem = reinterpret_cast<int *>(sGs + 9 * N);
    T *s_s2c = reinterpret_cast<T *>(s_nrem + N + (N & 1));
    unsigned *s_vm = reinterpret_cast<unsigned *>(smem_raw + a.off_vm);
    T *s_coef = reinterpret_cast<T *>(smem_raw + a.off_upart);        // [C][4] mode coefficients of q (and of v_k: MINRES), single frame
    T *svec = reinterpret_cast<T *>(smem_raw + a.off_vec);
    S2 *sspec = reinterpret_cast<S2 *>(smem_raw + a.off_spec);
    PairRef *ptab = reinterpret_cast<PairRef *>(smem_raw + a.off_ptab);
    UnitRec *s_unit = reinterpret_cast<UnitRec *>(smem_raw + a.off_unit);
    const int FB = BATCH ? a.fb : 1;                           // frames per slab pass
    constexpr bool MINRES = METHOD == METHOD_MINRES;
    constexpr int NVEC = MINRES ? 5 : 3;                                      // row vectors per unit in shared memory
    const int red_sz = (min(kPWarps / ((P + 31) >> 5), C) + (MINRES ? 4 : 2) * C) * P;      // partial sums of one frame (mac_slab)
    const int SCM = SC_HEAD + 2 * C + 3 * N, MRS = SCM + 2 * C;               // MINRES: channel sums of v, recurrence state
    C2 *Ubuf = work, *Vbuf = work + (size_t)FB * C * LD;      // [frame of the pass][c][LD] each
    const int NGS = a.ngs;
    C2 *bufA = work + (size_t)(gs < NGS ? gs : 0) * (P + LD), *bufB = bufA + P;   // row unit: natural [P], pass-1 result [LD]
    unsigned epoch = 0;
    const T half_n = (T)(0.5 * (n - 1)), dd = (T)a.g.d;
    int k = -2;                                      // iteration index seen by PSTAMP (no stamps outside the loop)
#define PSTAMP(pt) do { if (PROF) { if (a.dbg && tid == 0 && k >= 0) a.dbg[((size_t)b * a.n_iter + k) * PT_N + (pt)] = clock64(); } } while (0)
#define GRID_SYNC() do { epoch += G; grid_sync(a.flags, epoch); } while (0)

    // ---- slab ownership: CTA b owns k_x = b % Ph and a contiguous share of the frames
    // (the host balances the Ph x F slab passes over the CTAs: a CTA whose own share is below the average also takes
    // frames of ONE other slab, whose spectra it reads through L2; solve_persistent.cu: slab_segments)
    // The table row lives in shared memory and is re-read in every phase C, so that it holds no registers across phase R.
    const int kx = b % Ph;
    volatile int *s_seg = reinterpret_cast<volatile int *>(smem_raw + a.off_ms2 + (size_t)a.nq_m * P * sizeof(C2));
    if (tid < 8) s_seg[tid] = BATCH ? a.seg[b * 8 + tid] : (tid == 1 ? (b < Ph ? 1 : 0) : tid == 2 ? kx : 0);
    __syncthreads();
    const bool has_slab = (s_seg[1] - s_seg[0]) + (s_seg[4] - s_seg[3]) > 0;
    // slab thread maps
    const int c1 = tid / B, j2s = tid - c1 * B;      // pass 1: (channel, j2)
    const int c2s = tid / A, k1s = tid - c2s * A;    // pass 2: (channel, k1)
    // ---- row units of this CTA: ut = b + i G, i < nu; NGS of them per round, unit i0 + gs by the 16 lanes of group gs
    // single frame: strided (unit b + i G); batch: a contiguous chunk, so that a CTA's units belong to one or two frames and
    // it needs the modal sums of those frames only
    const int u_chunk = (F * U + G - 1) / G;
    const int u_base = BATCH ? b * u_chunk : b, u_stride = BATCH ? 1 : G;
    const int nu = BATCH ? max(0, min(u_chunk, F * U - u_base)) : ((b < F * U) ? (F * U - b + G - 1) / G : 0);
    const int fu_lo = BATCH ? min(u_base, F * U - 1) / U : 0, fu_n = BATCH ? (nu > 0 ? (u_base + nu - 1) / U - fu_lo + 1 : 0) : F;
    const int n_rounds = nu > 0 ? (nu + NGS - 1) / NGS : 1;

    for (int i = tid; i < P; i += kPThreads) tw[i] = a.tw[i];
    for (int i = tid; i < 9 * N; i += kPThreads) sGs[i] = a.g.Gs[i];
    for (int i = tid; i < N; i += kPThreads) s_nrem[i] = a.g.n_remove[i];
    for (int i = tid; i < C; i += kPThreads) s_s2c[i] = a.s2c[i];
    for (int i = tid; i < C * C; i += kPThreads) {
        const int oc = i / C, ci = i - oc * C, lo = min(oc, ci), hi = max(oc, ci);
        PairRef e;
        e.off = (lo * C - (lo * (lo - 1)) / 2 + hi - lo) * P;       // pair (c_out <= c_in); the transposed block is its conjugate
        e.sgn = ci < oc ? -1.f : 1.f;
        ptab[i] = e;
    }
    if (has_slab) {
        for (int q = 0; q < a.nq_m; ++q)
            for (int i = tid; i < P; i += kPThreads) {
                ms[q * P + i] = a.mspec[((size_t)q * Ph + kx) * P + i];
                ms2[q * P + i] = a.mspec[((size_t)q * Ph + s_seg[2]) * P + i];
            }
        if (a.spec_smem && s_seg[1] > s_seg[0]) {
            const S2 *gspec = a.spec + (size_t)kx * a.n_pair * P;
            for (int i = tid; i < a.n_pair * P; i += kPThreads) sspec[i] = gspec[i];
        }
    }
    for (int i = tid; i < F * SB; i += kPThreads) scal[i] = 0.0;
    for (int i = tid; i < nu * kGS; i += kPThreads) s_vm[i] = 0u;
    for (int i = tid; i < (nu > 0 ? nu : 1); i += kPThreads) {
        UnitRec u;
        const int ut = min(u_base + i * u_stride, F * U - 1);
        u.f = ut / U;
        const int uu = ut - u.f * U;
        u.c = uu / npairs; u.j = uu - u.c * npairs;
        u.s0 = a.g.row_ptr[2 * u.j]; u.s1 = a.g.row_ptr[2 * u.j + 1]; u.s2 = a.g.row_ptr[min(2 * u.j + 2, n)];
        u.pad0 = u.pad1 = 0;
        s_unit[i] = u;
    }
    __syncthreads();

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

    struct Unit { int f, c, j, comp, w, y0, s0, s1, s2; bool two; size_t vbase; };
    auto unit_of = [&](int i) {                      // from the table filled above
        const UnitRec u = s_unit[i];
        Unit q;
        q.f = u.f; q.c = u.c; q.j = u.j; q.comp = u.c & 1; q.w = u.c >> 1;
        q.y0 = 2 * u.j; q.two = q.y0 + 1 < n;
        q.s0 = u.s0; q.s1 = u.s1; q.s2 = u.s2;
        q.vbase = ((size_t)u.f * C + u.c) * nv;
        return q;
    };
    // dense rows (2 x n) of x, r, p, b of unit i
    auto dense = [&](int i, const Unit &q, int which) -> T * {
        if (a.vec_smem && which != 3) return svec + ((size_t)i * NVEC + (which < 3 ? which : which - 1)) * 2 * n;     // 4, 5: w_{k-1}, w_{k-2}
        T *base = which == 0 ? a.xd : which == 1 ? a.rd : which == 2 ? a.pd : which == 3 ? a.bd : which == 4 ? a.w1d : a.w2d;
        return base + (((size_t)q.f * C + q.c) * npad + q.y0) * n;
    };

    // one P-point transform bufA -> bufA by the 16 lanes of a row-unit group (all 32 lanes of the warp must call)
    // (nfill = number of leading elements of bufA that are stored; the rest count as zero)
    auto unit_fft = [&](bool act, int nfill) {
        __syncwarp();
        if (act && gl < B) dft_pass<T, A, true>(bufA + gl, B, (nfill - gl + B - 1) / B, bufB + gl, B + 1, tw, gl);
        __syncwarp();
        if (act && gl < A) dft_pass<T, B, false>(bufB + gl * (B + 1), 1, B, bufA + gl, A, tw, 0);
        __syncwarp();
    };
    // forward x-FFT of the two rows held in bufA (.x = row y0, .y = row y0+1; zero beyond n), split into the two
    // Hermitian half-spectra -> T1
    auto fwd_unit = [&](const Unit &q, bool act) {
        unit_fft(act, n);
        if (act) {
            C2 *out = a.T1 + (((size_t)q.f * Ph) * C + q.c) * npad + q.y0;
            constexpr int NLS = (Ph + kGS - 1) / kGS;          // every load before the first store
            C2 z1[NLS], z2[NLS];
#pragma unroll
            for (int m = 0; m < NLS; ++m) { const int kk = gl + m * kGS; if (kk < Ph) { z1[m] = bufA[kk]; z2[m] = bufA[kk == 0 ? 0 : P - kk]; } }
#pragma unroll
            for (int m = 0; m < NLS; ++m) {
                const int kk = gl + m * kGS;
                if (kk < Ph)
                    st_pair(out + (size_t)kk * C * npad, mk<T>((T)0.5 * (z1[m].x + z2[m].x), (T)0.5 * (z1[m].y - z2[m].y)),
                            q.two ? mk<T>((T)0.5 * (z1[m].y + z2[m].y), (T)-0.5 * (z1[m].x - z2[m].x)) : mk<T>((T)0, (T)0));
            }
        }
    };
    // ================================================================ init (A1: b = M_s s, Eq.33-34)
    // validity bits of the columns x = gl + 16 m each lane updates (bit row * 16 + m) and, for the mode removal, the
    // per-unit sums of s
    for (int i0 = 0; i0 < nu; i0 += NGS) {
        const int i = i0 + gs;
        const bool act = gs < NGS && i < nu;
        const Unit q = unit_of(act ? i : 0);
        double t0 = 0.0, t1 = 0.0;
        if (act) {
            for (int e = q.s0 + gl; e < q.s2; e += kGS) {
                const int row = e >= q.s1, xc = a.g.ix[e];
                atomicOr(&s_vm[i * kGS + (xc & (kGS - 1))], 1u << (row * 16 + xc / kGS));
                if (a.any_remove && a.mode != PM_STATE) {
                    const double v = (double)a.s_in[q.vbase + e];
                    const double coord = ((q.comp ? q.y0 + row : xc) - 0.5 * (n - 1)) * a.g.d;
                    t0 += v; t1 += coord * v;
                }
            }
        }
        __syncwarp();
        if (a.any_remove && a.mode != PM_STATE) {
            t0 = group_sum(t0); t1 = group_sum(t1);
            if (act && gl == 0) {
                const int u = (u_base + i * u_stride) - q.f * U;
                a.part_i[((size_t)q.f * U + u) * 2] = t0; a.part_i[((size_t)q.f * U + u) * 2 + 1] = t1;
            }
        }
    }
    if (a.any_remove && a.mode != PM_STATE) {
        GRID_SYNC();
        for (int item = warp; item < F * C * 2; item += NW) {
            const int f = item / (2 * C), rem = item - f * 2 * C, e = rem / C, c = rem - e * C;
            const double s = warp_sum_cg(a.part_i + ((size_t)f * U + c * npairs) * 2 + e, npairs, 2, lane);
            if (lane == 0) scal[f * SB + SC_HEAD + rem] = s;
        }
        __syncthreads();
        for (int t = tid; t < F * N; t += kPThreads) mode_coefs(t);
    }
    __syncthreads();
    for (int i0 = 0; i0 < nu; i0 += NGS) {
        const int i = i0 + gs;
        const bool act = gs < NGS && i < nu;
        const Unit q = unit_of(act ? i : 0);
        T *ux = dense(i, q, 0), *ur = dense(i, q, 1), *up = dense(i, q, 2), *ub = dense(i, q, 3);
        double rr = 0.0;
        __syncwarp();
        if (act) {
            for (int e = gl; e < 2 * n; e += kGS) { ux[e] = (T)0; ur[e] = (T)0; up[e] = (T)0; if (a.mode == PM_WARM) ub[e] = (T)0; }
            if (MINRES) { T *w1 = dense(i, q, 4), *w2 = dense(i, q, 5); for (int e = gl; e < 2 * n; e += kGS) { w1[e] = (T)0; w2[e] = (T)0; } }
            for (int e = gl; e < n; e += kGS) bufA[e] = mk<T>((T)0, (T)0);
        }
        __syncwarp();
        if (act) {
            const double *coef = scal + q.f * SB + SC_HEAD + 2 * C + q.w * 3;
            for (int e = q.s0 + gl; e < q.s2; e += kGS) {
                const int row = e >= q.s1, xc = a.g.ix[e], idx = row * n + xc;
                T fv;                                               // first transform: p_0 = b (cold), x0 (warm), p (state)
                if (a.mode == PM_STATE) {
                    ux[idx] = a.x[q.vbase + e]; ur[idx] = a.r[q.vbase + e]; fv = a.p[q.vbase + e]; up[idx] = fv;
                } else {
                    const double coord = ((q.comp ? q.y0 + row : xc) - 0.5 * (n - 1)) * a.g.d;
                    const T bv = (T)((double)a.s_in[q.vbase + e] - (coef[q.comp] + coef[2] * coord));   // b = s - Z a
                    if (a.mode == PM_WARM) { ub[idx] = bv; fv = (T)a.x0[q.vbase + e]; ux[idx] = fv; }
                    else { ur[idx] = bv; up[idx] = bv; fv = bv; rr += (double)bv * (double)bv; }         // cold: x = 0, r = p = b
                }
                if (row) bufA[xc].y = fv; else bufA[xc].x = fv;
            }
        }
        rr = group_sum(rr);
        if (act && gl == 0) a.part_r[u_base + i * u_stride] = rr;       // [f][unit]: unit index = f U + u
        fwd_unit(q, act);
    }
    GRID_SYNC();

    // MINRES: what one lane does per frame once |u_{kk-1}|^2 = uu is summed (kk = 0: |r0|^2): rotation kk-1 of the Lanczos
    // tridiagonal (oracle/solver.py:minres, same order), the coefficients of the pending x / w update, beta_kk for the product's
    // input, phibar^2 into the history.  Breakdowns freeze the iterate (reading G16 / G27).
    auto minres_scalars = [&](int f, int kk, double uu) {
        double *sc = scal + f * SB, *st = sc + MRS;
        if (kk == 0) {
            const double beta = sqrt(uu);
            st[MR_C] = -1.0; st[MR_S] = 0.0; st[MR_DBAR] = 0.0; st[MR_EPS] = 0.0; st[MR_PHIBAR] = beta;
            st[MR_FROZEN] = beta > 0.0 ? 0.0 : 1.0;
            st[MR_BETA] = beta; st[MR_INVBETA] = beta > 0.0 ? 1.0 / beta : 0.0; st[MR_PON] = 0.0;
            if (b == 0) a.hist[(size_t)f * a.hist_stride] = uu;
            return;
        }
        st[MR_PON] = 0.0;
        if (st[MR_FROZEN] == 0.0) {
            const double alpha = sc[SC_ALPHA], c = st[MR_C], s_ = st[MR_S], dbar = st[MR_DBAR], phibar = st[MR_PHIBAR];
            const double beta_next = sqrt(uu);
            const double delta = c * dbar + s_ * alpha, gbar = s_ * dbar - c * alpha;
            const double gamma = sqrt(gbar * gbar + beta_next * beta_next);
            if (!(gamma > 0.0)) {
                st[MR_FROZEN] = 1.0; st[MR_INVBETA] = 0.0;
            } else {
                const double c_new = gbar / gamma, s_new = beta_next / gamma;
                st[MR_PON] = 1.0; st[MR_PEPS] = st[MR_EPS]; st[MR_PDELTA] = delta; st[MR_PINVG] = 1.0 / gamma; st[MR_PPHI] = c_new * phibar;
                st[MR_PHIBAR] = s_new * phibar;
                st[MR_EPS] = s_ * beta_next; st[MR_DBAR] = -c * beta_next; st[MR_C] = c_new; st[MR_S] = s_new;
                st[MR_BETA] = beta_next;
                if (beta_next > 0.0) st[MR_INVBETA] = 1.0 / beta_next;
                else { st[MR_FROZEN] = 1.0; st[MR_INVBETA] = 0.0; }
            }
        }
        if (b == 0) a.hist[(size_t)f * a.hist_stride + kk] = st[MR_PHIBAR] * st[MR_PHIBAR];
    };

    // MINRES: alpha_k = v_k . M_s q = v.q - (Z^T v)^T (Z^T Z)^-1 Z^T q from the Parseval sums of one frame: one WFS term per
    // lane of a 16-lane group, summed in the group's fixed order (called by whole groups)
    auto minres_alpha = [&](const double *sc) {
        const double *S0 = sc + SC_HEAD, *S1 = S0 + C, *V0 = sc + SCM, *V1 = V0 + C;
        double term = 0.0;
        for (int i = gl; i < N; i += kGS) {
            const double tq[3] = {S0[2 * i], S0[2 * i + 1], S1[2 * i] + S1[2 * i + 1]}, tp[3] = {V0[2 * i], V0[2 * i + 1], V1[2 * i] + V1[2 * i + 1]};
            term += modal_quad(sGs + i * 9, tp, tq, s_nrem[i]);
        }
        return sc[SC_PQ] - group_sum(term);
    };

    // ================================================================ iterations (k = -1 is the warm-start product A x0)
    const int k_begin = (a.mode == PM_WARM) ? -1 : 0;
    const int n_t1 = C * npairs;                        // complex pairs in one T1 slab
    int voff[2];                                        // slab buffer offset c LD + y of the row pair e2 = tid + 512 m
    bool vtwo[2];
#pragma unroll
    for (int m = 0; m < 2; ++m) {
        const int e2 = tid + m * kPThreads, c = e2 / npairs, y = 2 * (e2 - c * npairs);
        voff[m] = c * LD + y; vtwo[m] = y + 1 < n;
    }
#pragma unroll 1
    for (k = k_begin; k < a.n_iter; ++k) {
        const bool pre = k < 0;
        const bool take_new = MINRES || pre || k == 0;  // p~ = T1 (p_0, or x0 for the warm-start product; MINRES: always, v_k = u_{k-1} / beta_k)
        PSTAMP(PT_START);
        // ---------------------------------------------------------- phase C: slab (kx, f)
        const int f_lo = BATCH ? s_seg[0] : 0, n_own = BATCH ? s_seg[1] - f_lo : (b < Ph ? 1 : 0), kx2 = BATCH ? s_seg[2] : kx;
        const int f2_lo = BATCH ? s_seg[3] : 0, n_items = BATCH ? n_own + s_seg[4] - f2_lo : n_own;
        C2 n0[2], n1[2], o0[2], o1[2];
        auto prefetch_slab = [&](int it, bool with_old) {
            const int f = it < n_own ? f_lo + it : f2_lo + (it - n_own), kxi = it < n_own ? kx : kx2;
            const C2 *t1 = a.T1 + ((size_t)f * Ph + kxi) * C * npad;
            const C2 *t1p = a.T1p + ((size_t)f * Ph + kxi) * C * npad;
#pragma unroll
            for (int m = 0; m < 2; ++m) {
                const int e2 = tid + m * kPThreads;
                if (e2 < n_t1) {
                    ldcg_pair(t1 + 2 * e2, n0[m], n1[m]);
                    if (with_old) ldcg_pair(t1p + 2 * e2, o0[m], o1[m]);
                }
            }
        };
        if (has_slab) prefetch_slab(0, !take_new);
        // scalars: rho_k, beta_k (one warp per frame, from the top warp down)
        if (!pre) {
            for (int f = NW - 1 - warp; f < F; f += NW) {
                double rho;
                if (k == 0 && a.mode == PM_STATE) rho = a.hist[(size_t)f * a.hist_stride];
                else rho = warp_sum_units(a.part_r + (size_t)f * U, U, lane);
                if (lane == 0) {
                    if (MINRES) {
                        minres_scalars(f, k, rho);
                    } else {
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
        }
        __syncthreads();
        PSTAMP(PT_RHO);
#pragma unroll 1
        for (int it = 0; it < n_items;) {
            const bool own = !BATCH || it < n_own;
            // batch: two consecutive frames of the same slab go through one pass together (the FFT passes are latency-bound
            // with 192 / 120 of the 512 threads busy: the second frame rides along)
            const int nf = (BATCH && FB == 2 && it + 1 < n_items && (it + 1 < n_own || it >= n_own)) ? 2 : 1;
            const int f0 = own ? f_lo + it : f2_lo + (it - n_own), kxi = own ? kx : kx2;
            const C2 *msi = own ? ms : ms2;
            const T wkx = (kxi == 0 || 2 * kxi == P) ? (T)1 : (T)2;
            if (!BATCH && it != 0) prefetch_slab(it, !take_new);     // (batch instance: issued before the previous pass's T2 store)
            // p~rows = r~rows + beta p~rows_old on rows 0..n-1 -> Vbuf[c][y] (the padding rows n..P-1 are never stored)
            for (int fr = 0; fr < nf; ++fr) {
                const int f = f0 + fr;
                const double *sc = scal + f * SB;
                const bool upd = !pre && sc[SC_UPD] != 0.0;
                const T beta = (T)sc[SC_BETA];
                C2 *t1p = a.T1p + ((size_t)f * Ph + kxi) * C * npad;
                C2 *Vf = Vbuf + (size_t)fr * C * LD;
                if (fr) prefetch_slab(it + fr, !take_new);
#pragma unroll
                for (int m = 0; m < 2; ++m) {
                    const int e2 = tid + m * kPThreads;
                    if (e2 < n_t1) {
                        C2 v0, v1;
                        if (take_new) {
                            v0 = n0[m]; v1 = n1[m];
                            if (MINRES && !pre) { const T ib = (T)sc[MRS + MR_INVBETA]; v0.x *= ib; v0.y *= ib; v1.x *= ib; v1.y *= ib; }
                        } else if (upd) { v0 = mk<T>(n0[m].x + beta * o0[m].x, n0[m].y + beta * o0[m].y); v1 = mk<T>(n1[m].x + beta * o1[m].x, n1[m].y + beta * o1[m].y); }
                        else { v0 = o0[m]; v1 = o1[m]; }
                        if (!MINRES && (take_new || upd)) st_pair(t1p + 2 * e2, v0, v1);
                        Vf[voff[m]] = v0;
                        if (vtwo[m]) Vf[voff[m] + 1] = v1;
                    }
                }
            }
            __syncthreads();
            PSTAMP(PT_BUILD);
            // forward y-FFT of the nf * C columns: pass 1 Vbuf -> Ubuf, pass 2 Ubuf -> Vbuf (natural k_y)
            const bool p1 = tid < nf * C * B, p2 = tid < nf * C * A;
            if (p1) dft_pass<T, A, true>(Vbuf + c1 * LD + j2s, B, (n - j2s + B - 1) / B, Ubuf + c1 * LD + j2s, B + 1, tw, j2s);
            __syncthreads();
            if (p2) dft_pass<T, B, false>(Ubuf + c2s * LD + k1s * (B + 1), 1, B, Vbuf + c2s * LD + k1s, A, tw, 0);
            __syncthreads();
            PSTAMP(PT_FFT);
#define TOMO_MAC(CT_, SP_) mac_slab<T, S, CT_, P, METHOD == METHOD_MINRES>(Vbuf + (size_t)fr * C * LD, Ubuf + (size_t)fr * C * LD, LD, SP_, ptab, msi, s_s2c, C, P, a.nq_m, a.any_remove, red + fr * red_sz, warp, lane)
#define TOMO_MAC_SWITCH(SP_)                                                               \
    switch (C) {                                                                           \
        case 4: TOMO_MAC(4, SP_); break;   case 6: TOMO_MAC(6, SP_); break;                \
        case 8: TOMO_MAC(8, SP_); break;   case 12: TOMO_MAC(12, SP_); break;              \
        case 16: TOMO_MAC(16, SP_); break; default: TOMO_MAC(0, SP_); break;               \
    }
#pragma unroll 1
            for (int fr = 0; fr < nf; ++fr) {
                if (a.spec_smem && own) { TOMO_MAC_SWITCH(sspec) } else { const S2 *gsp = a.spec + (size_t)kxi * a.n_pair * P; TOMO_MAC_SWITCH(gsp) }     // shared vs global loads
            }
#undef TOMO_MAC_SWITCH
#undef TOMO_MAC
            __syncthreads();
            PSTAMP(PT_MAC);
            // inverse y-FFT as a forward transform of conj(y~): pass 1 Ubuf -> Vbuf; the warps without pass-1 items
            // reduce the slab partials meanwhile
            // The warps without pass items reduce the slab partials meanwhile (from the top warp down): the first n_pub1 items beside
            // pass 1, the rest beside pass 2 (which keeps fewer warps busy), so that neither window holds more than ~one trip
            const int WPG = (P + 31) >> 5, Goc = min(NW / WPG, C);
            const int wb1 = (nf * C * B + 31) >> 5, wb2 = (nf * C * A + 31) >> 5;
            const int free1 = (!BATCH && NW - wb1 > 0) ? NW - wb1 : NW, free2 = (!BATCH && NW - wb2 > 0) ? NW - wb2 : NW;
            const int n_pub = nf * NQ, n_pub1 = (BATCH || n_pub <= free1) ? n_pub : max(free1, n_pub - free2);
            auto publish = [&](int lo, int hi, int nfree) {
                const int slot = NW - 1 - warp;
                if (slot < nfree) {
                    for (int tq = lo + slot; tq < hi; tq += nfree) {
                        const int fr = BATCH ? tq / NQ : 0, q1 = tq - fr * NQ;
                        const T *rd = red + fr * red_sz;
                        double s = 0.0;
                        if (q1 == 0) s = warp_sum_red<T>(rd, Goc * P, lane);
                        else if (a.any_remove) s = warp_sum_red<T>(rd + (Goc + q1 - 1) * P, P, lane);
                        if (lane == 0) a.part_s[((size_t)(f0 + fr) * NQ + q1) * Ph + kxi] = (double)wkx * s;
                    }
                }
            };
            if (p1) dft_pass<T, A, true>(Ubuf + c1 * LD + j2s, B, A, Vbuf + c1 * LD + j2s, B + 1, tw, j2s);
            publish(0, n_pub1, free1);
            __syncthreads();
            if (p2) dft_pass<T, B, false>(Vbuf + c2s * LD + k1s * (B + 1), 1, B, Ubuf + c2s * LD + k1s, A, tw, 0);
            publish(n_pub1, n_pub, free2);
            __syncthreads();
            // batch: the T1 / T1p loads of the next pass fly during this pass's T2 store
            if (BATCH && it + nf < n_items) prefetch_slab(it + nf, !take_new);
            // image rows y < n (conjugate back) -> T2[c][y / 2][kx][y & 1]
            for (int fr = 0; fr < nf; ++fr) {
                C2 *dst = a.T2 + (size_t)(f0 + fr) * C * npairs * Ph * 2 + (size_t)kxi * 2;
                const C2 *Uf = Ubuf + (size_t)fr * C * LD;
#pragma unroll
                for (int m = 0; m < 2; ++m) {
                    const int e = tid + m * kPThreads;
                    if (e < n_t1) {
                        const C2 u0 = Uf[voff[m]], u1 = vtwo[m] ? Uf[voff[m] + 1] : mk<T>((T)0, (T)0);
                        st_pair(dst + (size_t)e * Ph * 2, mk<T>(u0.x, -u0.y), mk<T>(u1.x, -u1.y));
                    }
                }
            }
            __syncthreads();
            it += nf;
        }
        PSTAMP(PT_INV);
        GRID_SYNC();
        PSTAMP(PT_BAR_B);
        // ---------------------------------------------------------- phase R: row units, NGS per round
#pragma unroll 1
        for (int rnd = 0; rnd < n_rounds; ++rnd) {
            const int i = rnd * NGS + gs;
            const bool act = gs < NGS && i < nu;
            const Unit q = unit_of(act ? i : 0);
            // stage 1 (no scalars needed): T2 -> conj(U + i V) with its Hermitian extension -> transform -> bufA[x] =
            // conj(row y0 + i row y0+1) of q = A p
            __syncwarp();
            if (act) {
                const C2 *src = a.T2 + (((size_t)q.f * C + q.c) * npairs + q.j) * Ph * 2;
                constexpr int NL = (Ph + kGS - 1) / kGS;                 // all loads in flight before the first use
                C2 u[NL], v[NL];
#pragma unroll
                for (int m = 0; m < NL; ++m) { const int kk = gl + m * kGS; if (kk < Ph) ldcg_pair(src + 2 * kk, u[m], v[m]); }
#pragma unroll
                for (int m = 0; m < NL; ++m) {
                    const int kk = gl + m * kGS;
                    if (kk < Ph) {
                        bufA[kk] = mk<T>(u[m].x - v[m].y, -(u[m].y + v[m].x));                               // conj(U_k + i V_k)
                        if (kk > 0 && 2 * kk < P) bufA[P - kk] = mk<T>(u[m].x + v[m].y, u[m].y - v[m].x);   // conj(conj(U_k) + i conj(V_k))
                    }
                }
            }
            if (rnd == 0) PSTAMP(PT_R_LOAD);
            unit_fft(act, P);
            if (rnd == 0) PSTAMP(PT_R_FFT1);
            if (rnd == 0) {
                // scalars: alpha_k, mode coefficients (reduction items from the top warps down)
                // (four items per trip, all their loads in flight at once: at batch 16 a warp has 13 items and one L2 round
                // trip per item cost 7.5 us)
                // items: p.q of every frame (alpha of the frames of the CTA's slab passes), then the modal sums of the frames
                // of its row units (batch: one or two frames; single frame: item = qq)
                constexpr int NLD = (Ph + 31) / 32, NB = BATCH ? 4 : MINRES ? 2 : 1;     // (MINRES has 1 + 2C(+2C) items: two per warp in one trip)
                // (MINRES: alpha_k of EVERY frame needs that frame's modal sums, for the rotation in the next phase C)
                const int n_sc = (BATCH && !MINRES) ? F + fu_n * (NQ - 1) : F * NQ;
                auto sc_item = [&](int item, int &f, int &qq) {
                    if (!BATCH || MINRES) { f = item / NQ; qq = item - f * NQ; }
                    else if (item < F) { f = item; qq = 0; }
                    else { const int r = item - F; f = fu_lo + r / (NQ - 1); qq = 1 + r % (NQ - 1); }
                };
                // single frame: the warps that hold no row unit this round take the items and, behind a barrier of their own, form
                // alpha_k and the mode coefficients of every channel (s_coef) while the unit warps are still in stage 1
                const int nuw = (min(NGS, nu) * kGS + 31) >> 5;             // warps with row units
                const bool split = !BATCH && MINRES && nuw + 2 <= NW;      // (CG: a row unit forms its few coefficients faster itself)
                const int NWs = split ? NW - nuw : NW;                      // warps that take items (from the top warp down)
                for (int item0 = NW - 1 - warp; item0 < n_sc && NW - 1 - warp < NWs; item0 += NB * NWs) {
                    double v[NB][NLD];
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        const int item = item0 + j * NWs;
                        int f = 0, qq = 0;
                        if (item < n_sc) sc_item(item, f, qq);
                        const bool on = item < n_sc && (qq == 0 || a.any_remove);
                        const double *src = a.part_s + ((size_t)f * NQ + qq) * Ph;
#pragma unroll
                        for (int m = 0; m < NLD; ++m) { const int i = lane + 32 * m; v[j][m] = (on && i < Ph) ? __ldcg(src + i) : 0.0; }
                    }
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        const int item = item0 + j * NWs;
                        if (item < n_sc) {
                            int f, qq;
                            sc_item(item, f, qq);
                            double t;
                            if constexpr (NLD == 5) t = ((v[j][0] + v[j][1]) + (v[j][2] + v[j][3])) + v[j][4];     // the order warp_sum_cg160 used
                            else { t = v[j][0]; for (int m = 1; m < NLD; ++m) t += v[j][m]; }
                            const double s = warp_sum(t);
                            const int nqs = C * (a.nq_m > 1 ? 2 : 1);             // modal sums of q, then (MINRES) of v
                            if (lane == 0) scal[f * SB + (qq == 0 ? SC_PQ : qq - 1 < nqs ? SC_HEAD + qq - 1 : SCM + qq - 1 - nqs)] = s;
                        }
                    }
                }
                if (split) {
                    if (warp >= nuw) {
                        asm volatile("bar.sync 1, %0;" ::"r"(NWs * 32) : "memory");
                        const double *sc = scal;
                        if (warp == NW - 1 && !pre) {                            // alpha_k (frame 0)
                            double al;
                            if (MINRES) al = minres_alpha(sc);
                            else { const double rho = sc[SC_RHO], pq = sc[SC_PQ]; al = (rho > 0.0 && pq > 0.0) ? div_as<T>(rho, pq) : 0.0; }   // breakdown: freeze (reading G16)
                            if (lane == 0) { scal[SC_ALPHA] = al; if (b == 0) a.alpha[0] = al; }
                        }
                        if (warp == NW - 2) for (int ch = lane; ch < C; ch += 32) {       // mode coefficients of channel ch (Eq.36)
                            const int w = ch >> 1, comp = ch & 1, nr = s_nrem[w];
                            const double *S0 = sc + SC_HEAD, *S1 = S0 + C;
                            const double tq[3] = {S0[2 * w], S0[2 * w + 1], S1[2 * w] + S1[2 * w + 1]};
                            double d0, d2;
                            modal_coef(sGs + w * 9, tq, nr, comp, d0, d2);
                            s_coef[ch * 4 + 0] = (comp < nr) ? (T)d0 : (T)0;
                            s_coef[ch * 4 + 1] = (2 < nr) ? (T)d2 : (T)0;
                            if (MINRES) {
                                const double *V0 = sc + SCM, *V1 = V0 + C;
                                const double tp[3] = {V0[2 * w], V0[2 * w + 1], V1[2 * w] + V1[2 * w + 1]};
                                modal_coef(sGs + w * 9, tp, nr, comp, d0, d2);
                                s_coef[ch * 4 + 2] = (comp < nr) ? (T)d0 : (T)0;
                                s_coef[ch * 4 + 3] = (2 < nr) ? (T)d2 : (T)0;
                            }
                        }
                    }
                }
                __syncthreads();
                // alpha_k is recorded for the next phase C / the tail; (batch, or too few free warps) every row unit derives alpha
                // and its own mode coefficients from the sums itself
                if (!pre && !split) {
                    if (MINRES && BATCH) {                                       // (single frame: recorded in stage 2 below)
                        for (int f0 = gs & ~1; f0 < F; f0 += kPThreads / kGS) {   // one 16-lane group per frame; the two groups of a
                            const int f = f0 + (gs & 1);                         // warp go through the full-mask shuffles together
                            double *sc = scal + min(f, F - 1) * SB;
                            const double al = minres_alpha(sc);
                            if (gl == 0 && f < F) { sc[SC_ALPHA] = al; if (b == 0) a.alpha[f] = al; }
                        }
                    } else if (!MINRES) {
                        for (int f = tid; f < F; f += kPThreads) {
                            double *sc = scal + f * SB;
                            const double rho = sc[SC_RHO], pq = sc[SC_PQ];
                            const double al = (rho > 0.0 && pq > 0.0) ? div_as<T>(rho, pq) : 0.0;     // breakdown: freeze (reading G16)
                            sc[SC_ALPHA] = al;
                            if (b == 0) a.alpha[f] = al;
                        }
                    }
                }
                PSTAMP(PT_SCAL);
            }
            // stage 2: q' = M_s q, CG vector updates, r.r partial, the new residual rows -> bufA -> forward x-FFT -> T1
            double rr = 0.0;
            double al_mr = 0.0;                      // MINRES: alpha_k of the unit's frame, one WFS term per lane of the group
            const int nuw2 = (min(NGS, nu) * kGS + 31) >> 5;
            const bool from_tab = !BATCH && MINRES && nuw2 + 2 <= NW;              // alpha and the coefficients were formed by the free warps
            if (MINRES && !pre) {
                if (from_tab) al_mr = scal[SC_ALPHA];
                else {
                    al_mr = minres_alpha(scal + q.f * SB);                       // (batch: bitwise the value recorded in SC_ALPHA above)
                    if (!BATCH && rnd == 0 && tid == 0) { scal[SC_ALPHA] = al_mr; if (b == 0) a.alpha[0] = al_mr; }
                }
            }
            if (act) {
                const double *sc = scal + q.f * SB;
                const double rho_k = sc[SC_RHO], pq_k = sc[SC_PQ];
                double al;
                if (from_tab) al = pre ? 0.0 : sc[SC_ALPHA];
                else al = (!pre && rho_k > 0.0 && pq_k > 0.0) ? div_as<T>(rho_k, pq_k) : 0.0;   // = sc[SC_ALPHA]
                const T alpha = (T)al, beta = (T)sc[SC_BETA];
                const bool apply = a.mode == PM_APPLY;
                const bool upd = sc[SC_UPD] != 0.0, step = al != 0.0 && !apply;
                // mode coefficients (Z^T Z)^-1 Z^T q of this unit's WFS from the channel sums (Eq.36)
                T c0 = (T)0, c2 = (T)0;
                if (from_tab) { c0 = s_coef[q.c * 4]; c2 = s_coef[q.c * 4 + 1]; }
                else {
                    const double *S0 = sc + SC_HEAD, *S1 = sc + SC_HEAD + C;
                    const double tq[3] = {S0[2 * q.w], S0[2 * q.w + 1], S1[2 * q.w] + S1[2 * q.w + 1]};
                    const int nr = s_nrem[q.w];
                    double d0, d2;
                    modal_coef(sGs + q.w * 9, tq, nr, q.comp, d0, d2);
                    c0 = (q.comp < nr) ? (T)d0 : (T)0;
                    c2 = (2 < nr) ? (T)d2 : (T)0;
                }
                const unsigned vm = s_vm[i * kGS + gl];
                const T *ub = dense(i, q, 3);

                // x, r, p of the unit: shared memory (vec_smem) or the dense global rows; separate code so that the
                // loads and stores are LDS/STS resp. LDG/STG, not generic
                auto update_rows = [&](T *ux, T *ur, T *up, const bool steady) {
                    constexpr int NX = (P / 2 + kGS) / kGS;              // columns per lane, n <= P/2 + 1
                    if (steady) {
                        // the steady-state iteration (k >= 1, no breakdown) on shared-memory rows, branch-free: every column x < n
                        // is processed; outside the pupil the rows hold zeros and stay zero (q is masked there: W_s), so the
                        // arithmetic of a valid element is that of the general code below, operation by operation
#pragma unroll
                        for (int m = 0; m < NX; ++m) {
                            const int xp = gl + m * kGS;
                            if (xp < n) {
                                const C2 z = bufA[xp];
                                T nr[2];
                                T rv_[2], pv_[2], xv_[2];        // the loads of both rows before the first store of the column
#pragma unroll
                                for (int row = 0; row < 2; ++row) { const int idx = row * n + xp; rv_[row] = ur[idx]; pv_[row] = up[idx]; xv_[row] = ux[idx]; }
#pragma unroll
                                for (int row = 0; row < 2; ++row) {
                                    const bool valid = (vm >> (row * 16 + m)) & 1u;
                                    const T coord = ((q.comp ? (T)(q.y0 + row) : (T)xp) - half_n) * dd;
                                    const T qm = (row ? -z.y : z.x) - (c0 + c2 * coord);
                                    const T qp = valid ? qm : (T)0;
                                    const int idx = row * n + xp;
                                    T rv = rv_[row];
                                    const T pv = rv + beta * pv_[row];
                                    up[idx] = pv;
                                    ux[idx] = xv_[row] + alpha * pv;
                                    rv -= alpha * qp;
                                    ur[idx] = rv;
                                    rr += (double)rv * (double)rv;
                                    nr[row] = rv;
                                }
                                bufA[xp] = mk<T>(nr[0], nr[1]);
                            }
                        }
                        return;
                    }
                    constexpr int NH = BATCH ? (NX + 1) / 2 : 1;         // two halves: every load of a half is issued before its
                                                                         // first store (a store between two loads serialises them:
                                                                         // one L2 round trip per element with the rows in global memory)
#pragma unroll
                    for (int h0 = 0; h0 < NX; h0 += NH) {
                        T rv_[NH][2], pv_[NH][2], xv_[NH][2];
#pragma unroll
                        for (int mm = 0; mm < NH; ++mm) {
                            const int m = h0 + mm, xp = gl + m * kGS;
#pragma unroll
                            for (int row = 0; row < 2; ++row) {
                                rv_[mm][row] = pv_[mm][row] = xv_[mm][row] = (T)0;
                                if (m < NX && xp < n && ((vm >> (row * 16 + m)) & 1u)) {
                                    const int idx = row * n + xp;
                                    if (pre) rv_[mm][row] = ub[idx];
                                    else { rv_[mm][row] = ur[idx]; pv_[mm][row] = up[idx]; xv_[mm][row] = ux[idx]; }
                                }
                            }
                        }
#pragma unroll
                        for (int mm = 0; mm < NH; ++mm) {
                            const int m = h0 + mm, xp = gl + m * kGS;
                            if (m < NX && xp < n) {
                                const C2 z = bufA[xp];
                                T nr[2] = {(T)0, (T)0};
#pragma unroll
                                for (int row = 0; row < 2; ++row) {
                                    if ((vm >> (row * 16 + m)) & 1u) {
                                        const T coord = ((q.comp ? (T)(q.y0 + row) : (T)xp) - half_n) * dd;
                                        const T qp = (row ? -z.y : z.x) - (c0 + c2 * coord);
                                        const int idx = row * n + xp;
                                        T rv;
                                        if (pre) {                                   // warm start: r = b - M_s q, p = r
                                            rv = rv_[mm][row] - qp;
                                            ur[idx] = rv; up[idx] = rv;
                                        } else if (apply) {                   // one product: r <- q' = M_s q
                                            rv = qp;
                                            ur[idx] = rv;
                                        } else {
                                            rv = rv_[mm][row];
                                            T pv = pv_[mm][row];
                                            if (upd) { pv = rv + beta * pv; up[idx] = pv; }
                                            if (step) {
                                                ux[idx] = xv_[mm][row] + alpha * pv;
                                                rv -= alpha * qp;
                                                ur[idx] = rv;
                                            }
                                        }
                                        rr += (double)rv * (double)rv;
                                        nr[row] = rv;
                                    }
                                }
                                bufA[xp] = mk<T>(nr[0], nr[1]);
                            }
                        }
                    }
                };
                // MINRES (one Lanczos step + the x / w update of the PREVIOUS iteration, whose rotation needed |u|): rows x, v_{k-1},
                // u_{k-1} (v_k = u_{k-1} / beta_k, re-projected: reading G27), w_{k-1}, w_{k-2}
                auto update_rows_mr = [&](T *ux, T *uvo, T *uvc, T *uw1, T *uw2, const bool steady_ok) {
                    const double *st = sc + MRS;
                    const bool frozen = st[MR_FROZEN] != 0.0, first = k == 0, pon = st[MR_PON] != 0.0;
                    const bool steady = steady_ok && !frozen && !first && pon;
                    const T alm = (T)al_mr, betak = (T)st[MR_BETA], ib = (T)st[MR_INVBETA];
                    const T peps = (T)st[MR_PEPS], pdelta = (T)st[MR_PDELTA], pinvg = (T)st[MR_PINVG], pphi = (T)st[MR_PPHI];
                    T cv0 = (T)0, cv2 = (T)0;                             // mode coefficients of v_k
                    if (from_tab) { cv0 = s_coef[q.c * 4 + 2]; cv2 = s_coef[q.c * 4 + 3]; }
                    else {
                        const double *V0 = sc + SCM, *V1 = V0 + C;
                        const double tp[3] = {V0[2 * q.w], V0[2 * q.w + 1], V1[2 * q.w] + V1[2 * q.w + 1]};
                        const int nr = s_nrem[q.w];
                        double d0, d2;
                        modal_coef(sGs + q.w * 9, tp, nr, q.comp, d0, d2);
                        cv0 = (q.comp < nr) ? (T)d0 : (T)0;
                        cv2 = (2 < nr) ? (T)d2 : (T)0;
                    }
                    constexpr int NX = (P / 2 + kGS) / kGS;              // columns per lane
                    if (steady) {
                        // the steady-state iteration (k >= 1, a pending x / w update, no breakdown) on shared-memory rows, branch-free as
                        // in update_rows: outside the pupil the five rows hold zeros and stay zero (q and the projection of v_k are
                        // masked there); a valid element goes through the operations of the general code below
#pragma unroll
                        for (int m = 0; m < NX; ++m) {
                            const int xp = gl + m * kGS;
                            if (xp < n) {
                                const C2 z = bufA[xp];
                                T nr[2];
                                T vo_[2], w1_[2], w2_[2], xv_[2], vc_[2];        // the loads of both rows before the first store of the column
#pragma unroll
                                for (int row = 0; row < 2; ++row) {
                                    const int idx = row * n + xp;
                                    vo_[row] = uvo[idx]; w1_[row] = uw1[idx]; w2_[row] = uw2[idx]; xv_[row] = ux[idx]; vc_[row] = uvc[idx];
                                }
#pragma unroll
                                for (int row = 0; row < 2; ++row) {
                                    const bool valid = (vm >> (row * 16 + m)) & 1u;
                                    const int idx = row * n + xp;
                                    const T coord = ((q.comp ? (T)(q.y0 + row) : (T)xp) - half_n) * dd;
                                    const T vo = vo_[row];
                                    const T w1v = w1_[row];
                                    const T w = (vo - peps * w2_[row] - pdelta * w1v) * pinvg;
                                    ux[idx] = xv_[row] + pphi * w;
                                    uw2[idx] = w1v; uw1[idx] = w;
                                    const T vpm = vc_[row] * ib - (cv0 + cv2 * coord);
                                    const T qm = (row ? -z.y : z.x) - (c0 + c2 * coord);
                                    const T vp = valid ? vpm : (T)0, qp = valid ? qm : (T)0;
                                    const T uv = qp - alm * vp - betak * vo;
                                    uvo[idx] = vp; uvc[idx] = uv;
                                    rr += (double)uv * (double)uv;
                                    nr[row] = uv;
                                }
                                bufA[xp] = mk<T>(nr[0], nr[1]);
                            }
                        }
                        return;
                    }
                    constexpr int NH = (NX + 1) / 2;                     // two halves (five vectors: all columns at once spill);
                                                                         // every load of a half is issued before its first store
#pragma unroll
                    for (int h0 = 0; h0 < NX; h0 += NH) {
                        T vo_[NH][2], vc_[NH][2], w1_[NH][2], w2_[NH][2], xv_[NH][2];
#pragma unroll
                        for (int mm = 0; mm < NH; ++mm) {
                            const int m = h0 + mm, xp = gl + m * kGS;
#pragma unroll
                            for (int row = 0; row < 2; ++row) {
                                vo_[mm][row] = vc_[mm][row] = w1_[mm][row] = w2_[mm][row] = xv_[mm][row] = (T)0;
                                if (m < NX && xp < n && ((vm >> (row * 16 + m)) & 1u)) {
                                    const int idx = row * n + xp;
                                    if (!first) vo_[mm][row] = uvo[idx];
                                    vc_[mm][row] = uvc[idx];
                                    if (pon) { w1_[mm][row] = uw1[idx]; w2_[mm][row] = uw2[idx]; xv_[mm][row] = ux[idx]; }
                                }
                            }
                        }
#pragma unroll
                        for (int mm = 0; mm < NH; ++mm) {
                            const int m = h0 + mm, xp = gl + m * kGS;
                            if (m < NX && xp < n) {
                                const C2 z = bufA[xp];
                                T nr[2] = {(T)0, (T)0};
#pragma unroll
                                for (int row = 0; row < 2; ++row) {
                                    if ((vm >> (row * 16 + m)) & 1u) {
                                        const int idx = row * n + xp;
                                        const T coord = ((q.comp ? (T)(q.y0 + row) : (T)xp) - half_n) * dd;
                                        const T vo = vo_[mm][row];
                                        if (pon) {
                                            const T w = (vo - peps * w2_[mm][row] - pdelta * w1_[mm][row]) * pinvg;
                                            ux[idx] = xv_[mm][row] + pphi * w;
                                            uw2[idx] = w1_[mm][row]; uw1[idx] = w;
                                        }
                                        if (!frozen) {
                                            const T vp = vc_[mm][row] * ib - (cv0 + cv2 * coord);
                                            const T qp = (row ? -z.y : z.x) - (c0 + c2 * coord);
                                            const T uv = qp - alm * vp - betak * vo;
                                            uvo[idx] = vp; uvc[idx] = uv;
                                            rr += (double)uv * (double)uv;
                                            nr[row] = uv;
                                        }
                                    }
                                }
                                bufA[xp] = mk<T>(nr[0], nr[1]);
                            }
                        }
                    }
                };
                if (MINRES && !pre) {
                    if (a.vec_smem) {
                        T *base = svec + (size_t)i * NVEC * 2 * n;
                        update_rows_mr(base, base + 2 * n, base + 4 * n, base + 6 * n, base + 8 * n, true);
                    } else {
                        const size_t o = (((size_t)q.f * C + q.c) * npad + q.y0) * n;
                        update_rows_mr(a.xd + o, a.rd + o, a.pd + o, a.w1d + o, a.w2d + o, false);
                    }
                } else if (a.vec_smem) {
                    T *base = svec + (size_t)i * NVEC * 2 * n;
                    update_rows(base, base + 2 * n, base + 4 * n, !pre && !apply && upd && step);
                } else {
                    const size_t o = (((size_t)q.f * C + q.c) * npad + q.y0) * n;
                    update_rows(a.xd + o, a.rd + o, a.pd + o, false);
                }
            }
            rr = group_sum(rr);
            if (act && gl == 0) a.part_r[u_base + i * u_stride] = rr;       // [f][unit]: unit index = f U + u
            if (rnd == 0) PSTAMP(PT_R_UPD);
            fwd_unit(q, act);
            if (rnd == 0) PSTAMP(PT_R_FFT2);
        }
        PSTAMP(PT_ROWS);
        GRID_SYNC();
        PSTAMP(PT_BAR_A);
    }
    k = -2;

    // ================================================================ tail: rho_{n_iter}; optional p = r + beta p; x, r, p -> valid-only layout
    // (MINRES: the last rotation and the pending x update)
    for (int f = NW - 1 - warp; f < F; f += NW) {
        double rho;
        if (a.n_iter == 0 && a.mode == PM_STATE) rho = a.hist[(size_t)f * a.hist_stride];
        else rho = warp_sum_units(a.part_r + (size_t)f * U, U, lane);
        if (lane == 0) {
            if (MINRES) {
                minres_scalars(f, a.n_iter, rho);
            } else {
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
    }
    __syncthreads();
    for (int i0 = 0; i0 < nu; i0 += NGS) {
        const int i = i0 + gs;
        if (gs >= NGS || i >= nu) continue;
        const Unit q = unit_of(i);
        const double *sc = scal + q.f * SB;
        const bool fin = !MINRES && a.finalize_p && sc[SC_UPD] != 0.0;
        const T beta = (T)sc[SC_BETA];
        const T *ux = dense(i, q, 0), *ur = dense(i, q, 1), *up = dense(i, q, 2);
        const double *st = sc + MRS;
        const bool pon = MINRES && st[MR_PON] != 0.0;
        const T peps = pon ? (T)st[MR_PEPS] : (T)0, pdelta = pon ? (T)st[MR_PDELTA] : (T)0, pinvg = pon ? (T)st[MR_PINVG] : (T)0,
                pphi = pon ? (T)st[MR_PPHI] : (T)0;
        const T *uw1 = MINRES ? dense(i, q, 4) : ux, *uw2 = MINRES ? dense(i, q, 5) : ux;
        for (int e = q.s0 + gl; e < q.s2; e += kGS) {
            const int row = e >= q.s1, idx = row * n + a.g.ix[e];
            T pv = up[idx], xv = ux[idx];
            const T rv = ur[idx];
            if (fin) pv = rv + beta * pv;
            if (pon) xv += pphi * ((rv - peps * uw2[idx] - pdelta * uw1[idx]) * pinvg);      // x_n = x_{n-1} + phi_n w_n, w_n from v_n = rv
            a.x[q.vbase + e] = xv; a.r[q.vbase + e] = rv; a.p[q.vbase + e] = pv;
        }
    }
#undef PSTAMP
#undef GRID_SYNC
}

}  // namespace tomo
