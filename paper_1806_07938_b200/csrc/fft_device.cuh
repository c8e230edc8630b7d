// fft_device.cuh -- warp-cooperative shared-memory FFT of 5-smooth length for sm_100a.
//
// One warp transforms one complex sequence of length P held in shared memory by the Stockham autosort
// algorithm: passes of radix 8/4/2/5/3, ping-ponging between two P-element buffers, __syncwarp between passes
// (no block barrier), twiddles exp(-2 pi i t/P) from a shared-memory table.  This is steps 2 and 4 of the
// paper's 2RBT product (Eq.21, Eq.23) in its 2-D separable form (reading G10).
#pragma once
// The header also compiles as plain C++ (g++, no CUDA) with NL = 1 so that tests/ can check every radix and
// length on the CPU box; on the device NL = 32 lanes share one transform.
#if defined(__CUDACC__)
#include <cuda_runtime.h>
#define TOMO_HD __host__ __device__ __forceinline__
#else
#define TOMO_HD inline
#ifndef TOMO_HOST_VEC_TYPES
#define TOMO_HOST_VEC_TYPES
struct float2 { float x, y; };
struct double2 { double x, y; };
#endif
#define __restrict__
#endif

namespace tomo {

template <typename T> struct cx_of;
template <> struct cx_of<float> { typedef float2 type; };
template <> struct cx_of<double> { typedef double2 type; };

template <typename T> TOMO_HD typename cx_of<T>::type mk(T a, T b) {
    typename cx_of<T>::type r; r.x = a; r.y = b; return r;
}
template <typename C> TOMO_HD C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> TOMO_HD C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename C> TOMO_HD C cmul(C a, C b) {
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
template <typename C> TOMO_HD C cmulc(C a, C b) {   // a * conj(b)
    C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r;
}
// multiply by -i (forward) or +i (inverse)
template <bool INV, typename C> TOMO_HD C rot90(C a) {
    C r;
    if (INV) { r.x = -a.y; r.y = a.x; } else { r.x = a.y; r.y = -a.x; }
    return r;
}

struct FftDesc {          // filled on the host, passed by value
    int P;                // length
    int nrad;             // number of passes
    int rad[8];           // radix of each pass, product = P
};

// ---------------------------------------------------------------------------------------------- small DFTs
// b_k = sum_j a_j w^{jk}, w = exp(-+2 pi i / R); in place on a register array.
template <typename T, int R, bool INV> struct SmallDft;

template <typename T, bool INV> struct SmallDft<T, 2, INV> {
    typedef typename cx_of<T>::type C;
    TOMO_HD static void run(C *v) { C a = v[0], b = v[1]; v[0] = cadd(a, b); v[1] = csub(a, b); }
};

template <typename T, bool INV> struct SmallDft<T, 4, INV> {
    typedef typename cx_of<T>::type C;
    TOMO_HD static void run(C *v) {
        C s0 = cadd(v[0], v[2]), d0 = csub(v[0], v[2]);
        C s1 = cadd(v[1], v[3]), d1 = rot90<INV>(csub(v[1], v[3]));
        v[0] = cadd(s0, s1); v[2] = csub(s0, s1);
        v[1] = cadd(d0, d1); v[3] = csub(d0, d1);
    }
};

template <typename T, bool INV> struct SmallDft<T, 8, INV> {
    typedef typename cx_of<T>::type C;
    TOMO_HD static void run(C *v) {
        const T h = (T)0.70710678118654752440;
        C e[4] = {v[0], v[2], v[4], v[6]}, o[4] = {v[1], v[3], v[5], v[7]};
        SmallDft<T, 4, INV>::run(e);
        SmallDft<T, 4, INV>::run(o);
        // o_k *= w8^k
        C t1, t3;
        if (INV) { t1 = mk<T>(h * (o[1].x - o[1].y), h * (o[1].x + o[1].y)); t3 = mk<T>(-h * (o[3].x + o[3].y), h * (o[3].x - o[3].y)); }
        else     { t1 = mk<T>(h * (o[1].x + o[1].y), h * (o[1].y - o[1].x)); t3 = mk<T>(h * (o[3].y - o[3].x), -h * (o[3].x + o[3].y)); }
        C t2 = rot90<INV>(o[2]);
        v[0] = cadd(e[0], o[0]); v[4] = csub(e[0], o[0]);
        v[1] = cadd(e[1], t1);   v[5] = csub(e[1], t1);
        v[2] = cadd(e[2], t2);   v[6] = csub(e[2], t2);
        v[3] = cadd(e[3], t3);   v[7] = csub(e[3], t3);
    }
};

template <typename T, bool INV> struct SmallDft<T, 3, INV> {
    typedef typename cx_of<T>::type C;
    TOMO_HD static void run(C *v) {
        const T s = (T)0.86602540378443864676;            // sin(2 pi/3)
        C t = cadd(v[1], v[2]);
        C m = mk<T>(v[0].x - (T)0.5 * t.x, v[0].y - (T)0.5 * t.y);
        C d = csub(v[1], v[2]);
        C r = rot90<INV>(mk<T>(s * d.x, s * d.y));        // -+ i s (v1 - v2)
        v[0] = cadd(v[0], t); v[1] = cadd(m, r); v[2] = csub(m, r);
    }
};

template <typename T, bool INV> struct SmallDft<T, 5, INV> {
    typedef typename cx_of<T>::type C;
    TOMO_HD static void run(C *v) {
        const T c1 = (T)0.30901699437494742410, c2 = (T)-0.80901699437494742410;   // cos(2pi/5), cos(4pi/5)
        const T s1 = (T)0.95105651629515357212, s2 = (T)0.58778525229247312917;    // sin(2pi/5), sin(4pi/5)
        C a1 = cadd(v[1], v[4]), b1 = csub(v[1], v[4]);
        C a2 = cadd(v[2], v[3]), b2 = csub(v[2], v[3]);
        C m1 = mk<T>(v[0].x + c1 * a1.x + c2 * a2.x, v[0].y + c1 * a1.y + c2 * a2.y);
        C m2 = mk<T>(v[0].x + c2 * a1.x + c1 * a2.x, v[0].y + c2 * a1.y + c1 * a2.y);
        C r1 = rot90<INV>(mk<T>(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y));
        C r2 = rot90<INV>(mk<T>(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y));
        v[0] = cadd(v[0], cadd(a1, a2));
        v[1] = cadd(m1, r1); v[4] = csub(m1, r1);
        v[2] = cadd(m2, r2); v[3] = csub(m2, r2);
    }
};

// ---------------------------------------------------------------------------------------------- one pass
// Stockham DIF pass: ncur = current sub-length, s = stride (product of the radices already done), m = ncur/R,
//   y[q + s (R p + k)] = w_ncur^{p k} sum_j x[q + s (p + m j)] w_R^{jk},   p < m, q < s.
template <typename T, int R, bool INV, int NL>
TOMO_HD void fft_pass(const typename cx_of<T>::type *__restrict__ x,
                                         typename cx_of<T>::type *__restrict__ y, int P, int s, int ncur,
                                         const typename cx_of<T>::type *__restrict__ tw, int lane) {
    typedef typename cx_of<T>::type C;
    const int nb = P / R;                      // butterflies in this pass; s * m == nb
    const bool last = (ncur == R);
    for (int idx = lane; idx < nb; idx += NL) {
        const int p = idx / s, q = idx - p * s;
        C v[R];
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = x[idx + nb * j];
        SmallDft<T, R, INV>::run(v);
        C *out = y + q + s * R * p;
        out[0] = v[0];
        if (last) {
#pragma unroll
            for (int k = 1; k < R; ++k) out[s * k] = v[k];
        } else {
            const int t = p * s;               // w_ncur^p = w_P^{p s}
#pragma unroll
            for (int k = 1; k < R; ++k) {
                const C w = tw[t * k];
                out[s * k] = INV ? cmulc(v[k], w) : cmul(v[k], w);
            }
        }
    }
}

// Transform `a` (length d.P) using `b` as the second buffer; returns the buffer that holds the result.
// All NL lanes of the warp must call it; the warp-level fence after filling `a` is done here; the caller
// must not touch either buffer until it returns.
template <typename T, bool INV, int NL = 32>
TOMO_HD typename cx_of<T>::type *warp_fft(typename cx_of<T>::type *a, typename cx_of<T>::type *b,
                                                            const FftDesc &d,
                                                            const typename cx_of<T>::type *__restrict__ tw, int lane) {
    typedef typename cx_of<T>::type C;
    C *x = a, *y = b;
    int s = 1, ncur = d.P;
#ifdef __CUDA_ARCH__
    __syncwarp();
#endif
    for (int i = 0; i < d.nrad; ++i) {
        const int R = d.rad[i];
        switch (R) {
            case 8: fft_pass<T, 8, INV, NL>(x, y, d.P, s, ncur, tw, lane); break;
            case 4: fft_pass<T, 4, INV, NL>(x, y, d.P, s, ncur, tw, lane); break;
            case 5: fft_pass<T, 5, INV, NL>(x, y, d.P, s, ncur, tw, lane); break;
            case 3: fft_pass<T, 3, INV, NL>(x, y, d.P, s, ncur, tw, lane); break;
            default: fft_pass<T, 2, INV, NL>(x, y, d.P, s, ncur, tw, lane); break;
        }
        ncur /= R; s *= R;
        C *t = x; x = y; y = t;
#ifdef __CUDA_ARCH__
        __syncwarp();
#endif
    }
    return x;
}

// ---------------------------------------------------------------------------------------------- compile-time plan
// Same Stockham passes with the length, strides and trip counts known at compile time (no integer division, fully
// unrolled); radix order as plan_fft on the host: 5s, 3s, 8s, 4s, 2s.
template <int N> struct PickRadix {
    static constexpr int value = (N % 5 == 0) ? 5 : (N % 3 == 0) ? 3 : (N % 8 == 0) ? 8 : (N % 4 == 0) ? 4 : 2;
};
template <int N> struct CountPasses { static constexpr int value = 1 + CountPasses<N / PickRadix<N>::value>::value; };
template <> struct CountPasses<1> { static constexpr int value = 0; };

template <typename T, int R, bool INV, int P, int S, int NCUR, int NL>
TOMO_HD void fft_pass_static(const typename cx_of<T>::type *__restrict__ x, typename cx_of<T>::type *__restrict__ y,
                             const typename cx_of<T>::type *__restrict__ tw, int lane) {
    typedef typename cx_of<T>::type C;
    constexpr int nb = P / R;
    constexpr bool last = (NCUR == R);
    constexpr int trips = (nb + NL - 1) / NL;
#pragma unroll
    for (int it = 0; it < trips; ++it) {
        const int idx = lane + it * NL;
        if ((nb % NL == 0) || idx < nb) {
            const int p = idx / S, q = idx - p * S;
            C v[R];
#pragma unroll
            for (int j = 0; j < R; ++j) v[j] = x[idx + nb * j];
            SmallDft<T, R, INV>::run(v);
            C *out = y + q + S * R * p;
            out[0] = v[0];
            if (last) {
#pragma unroll
                for (int k = 1; k < R; ++k) out[S * k] = v[k];
            } else {
                const int t = p * S;
#pragma unroll
                for (int k = 1; k < R; ++k) {
                    const C w = tw[t * k];
                    out[S * k] = INV ? cmulc(v[k], w) : cmul(v[k], w);
                }
            }
        }
    }
}

template <typename T, bool INV, int P, int S, int NCUR, int NL> struct FftChain {
    typedef typename cx_of<T>::type C;
    TOMO_HD static C *run(C *x, C *y, const C *tw, int lane) {
        constexpr int R = PickRadix<NCUR>::value;
        fft_pass_static<T, R, INV, P, S, NCUR, NL>(x, y, tw, lane);
#ifdef __CUDA_ARCH__
        __syncwarp();
#endif
        return FftChain<T, INV, P, S * R, NCUR / R, NL>::run(y, x, tw, lane);
    }
};
template <typename T, bool INV, int P, int S, int NL> struct FftChain<T, INV, P, S, 1, NL> {
    typedef typename cx_of<T>::type C;
    TOMO_HD static C *run(C *x, C *, const C *, int) { return x; }
};

// Compile-time-planned counterpart of warp_fft: same contract, same result buffer.
template <typename T, bool INV, int P, int NL = 32>
TOMO_HD typename cx_of<T>::type *warp_fft_static(typename cx_of<T>::type *a, typename cx_of<T>::type *b,
                                                 const typename cx_of<T>::type *tw, int lane) {
#ifdef __CUDA_ARCH__
    __syncwarp();
#endif
    return FftChain<T, INV, P, 1, P, NL>::run(a, b, tw, lane);
}

}  // namespace tomo
