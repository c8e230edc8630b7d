// fft_reg.cuh -- register-resident two-pass FFT building blocks for sm_100a.
//
// A length-P transform (steps 2 and 4 of the paper's 2RBT product, Eq.21 L224 / Eq.23, in the 2-D
// separable form of reading G10) is split P = R * M and done by two groups of threads that each hold one small
// DFT entirely in registers, with ONE shared-memory exchange in between:
//
//   input index  j = j1 * M + j2   (j1 < R, j2 < M)          output index  k = k1 + R * k2   (k1 < R, k2 < M)
//   pass 1, thread j2 (M threads):  Y[k1][j2] = W_P^{j2 k1} * sum_j1 x[j1 M + j2] W_R^{j1 k1}      (radix R)
//   pass 2, thread k1 (R threads):  X[k1 + R k2] = sum_j2 Y[k1][j2] W_M^{j2 k2}                     (radix M)
//
// Small DFTs: 2, 3, 4, 5, 8 from fft_device.cuh; 16 = 4 x 4 with explicit twiddles; 6, 10, 12, 15, 20 by the
// prime-factor (Good-Thomas) map, which needs no twiddles.  The header also compiles as plain C++ for the CPU tests.
#pragma once
#include "fft_device.cuh"

namespace tomo {

// ---------------------------------------------------------------------------------------------- radix 16 = 4 x 4
template <typename T, bool INV> struct SmallDft<T, 16, INV> {
    typedef typename cx_of<T>::type C;
    // multiply by W16^t (forward) or its conjugate (inverse), t a compile-time constant
    template <int t> TOMO_HD static C tw16(C a) {
        const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173, h = (T)0.70710678118654752440;
        // W16^t = (cr, -ci) forward, (cr, +ci) inverse
        constexpr int q = t % 16;
        T cr, ci;
        if (q == 0) return a;
        else if (q == 1) { cr = c1; ci = s1; }
        else if (q == 2) { cr = h; ci = h; }
        else if (q == 3) { cr = s1; ci = c1; }
        else if (q == 4) return rot90<INV>(a);
        else if (q == 6) { cr = -h; ci = h; }
        else if (q == 9) { cr = -c1; ci = -s1; }
        else { cr = (T)1; ci = (T)0; }
        const T wi = INV ? ci : -ci;
        return mk<T>(a.x * cr - a.y * wi, a.x * wi + a.y * cr);
    }
    TOMO_HD static void run(C *v) {
        // step 1: four radix-4 DFTs over j1 (stride 4), twiddle W16^{j2 k1}
        C c0[4] = {v[0], v[4], v[8], v[12]}, c1[4] = {v[1], v[5], v[9], v[13]};
        C c2[4] = {v[2], v[6], v[10], v[14]}, c3[4] = {v[3], v[7], v[11], v[15]};
        SmallDft<T, 4, INV>::run(c0); SmallDft<T, 4, INV>::run(c1);
        SmallDft<T, 4, INV>::run(c2); SmallDft<T, 4, INV>::run(c3);
        c1[1] = tw16<1>(c1[1]); c1[2] = tw16<2>(c1[2]); c1[3] = tw16<3>(c1[3]);
        c2[1] = tw16<2>(c2[1]); c2[2] = tw16<4>(c2[2]); c2[3] = tw16<6>(c2[3]);
        c3[1] = tw16<3>(c3[1]); c3[2] = tw16<6>(c3[2]); c3[3] = tw16<9>(c3[3]);
        // step 2: for each k1 a radix-4 DFT over j2 -> X[k1 + 4 k2]
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) {
            C t[4] = {c0[k1], c1[k1], c2[k1], c3[k1]};
            SmallDft<T, 4, INV>::run(t);
            v[k1] = t[0]; v[k1 + 4] = t[1]; v[k1 + 8] = t[2]; v[k1 + 12] = t[3];
        }
    }
};

// ---------------------------------------------------------------------------------------------- prime-factor DFTs
// R = R1 * R2 with gcd(R1, R2) = 1:  j = (R2 j1 + R1 j2) mod R,  k = (R2 a k1 + R1 b k2) mod R,
// a = R2^-1 mod R1, b = R1^-1 mod R2  =>  X[k] = sum x[j] W_R1^{j1 k1} W_R2^{j2 k2}: no twiddle factors.
template <int A, int M> struct ModInv {
    static constexpr int calc() { for (int i = 1; i < M; ++i) if ((A * i) % M == 1) return i; return 1; }
    static constexpr int value = calc();
};
template <typename T, int R1, int R2, bool INV> struct PfaDft {
    typedef typename cx_of<T>::type C;
    TOMO_HD static void run(C *v) {
        constexpr int R = R1 * R2;
        constexpr int a = ModInv<R2 % R1, R1>::value, b = ModInv<R1 % R2, R2>::value;
        C w[R];
#pragma unroll
        for (int j2 = 0; j2 < R2; ++j2) {
            C t[R1];
#pragma unroll
            for (int j1 = 0; j1 < R1; ++j1) t[j1] = v[(R2 * j1 + R1 * j2) % R];
            SmallDft<T, R1, INV>::run(t);
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) w[k1 * R2 + j2] = t[k1];
        }
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) {
            C t[R2];
#pragma unroll
            for (int j2 = 0; j2 < R2; ++j2) t[j2] = w[k1 * R2 + j2];
            SmallDft<T, R2, INV>::run(t);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) v[(R2 * a * k1 + R1 * b * k2) % R] = t[k2];
        }
    }
};
template <typename T, bool INV> struct SmallDft<T, 6, INV> : PfaDft<T, 2, 3, INV> {};
template <typename T, bool INV> struct SmallDft<T, 10, INV> : PfaDft<T, 2, 5, INV> {};
template <typename T, bool INV> struct SmallDft<T, 12, INV> : PfaDft<T, 3, 4, INV> {};
template <typename T, bool INV> struct SmallDft<T, 15, INV> : PfaDft<T, 3, 5, INV> {};
template <typename T, bool INV> struct SmallDft<T, 20, INV> : PfaDft<T, 4, 5, INV> {};

// ---------------------------------------------------------------------------------------------- two-pass split
// P = A * B, A <= B <= 16 (or 20): the sizes the persistent kernel is instantiated for.
template <int P> struct Fact2 { static constexpr int A = 0, B = 0; };
#define TOMO_FACT2(P_, A_, B_) template <> struct Fact2<P_> { static constexpr int A = A_, B = B_; }
TOMO_FACT2(16, 4, 4);    TOMO_FACT2(20, 4, 5);    TOMO_FACT2(24, 3, 8);    TOMO_FACT2(32, 4, 8);   TOMO_FACT2(40, 5, 8);
TOMO_FACT2(48, 6, 8);    TOMO_FACT2(64, 8, 8);    TOMO_FACT2(80, 8, 10);   TOMO_FACT2(128, 8, 16); TOMO_FACT2(160, 10, 16);
TOMO_FACT2(180, 12, 15); TOMO_FACT2(192, 12, 16); TOMO_FACT2(240, 15, 16); TOMO_FACT2(256, 16, 16); TOMO_FACT2(320, 16, 20);
#undef TOMO_FACT2
// run-time view of the same table (host side: shared-memory sizing); returns false if P has no split
inline bool fact2_of(int P, int *A, int *B) {
    switch (P) {
#define TOMO_F2CASE(P_) case P_: *A = Fact2<P_>::A; *B = Fact2<P_>::B; return true
        TOMO_F2CASE(16); TOMO_F2CASE(20); TOMO_F2CASE(24); TOMO_F2CASE(32); TOMO_F2CASE(40); TOMO_F2CASE(48); TOMO_F2CASE(64);
        TOMO_F2CASE(80); TOMO_F2CASE(128); TOMO_F2CASE(160); TOMO_F2CASE(180); TOMO_F2CASE(192); TOMO_F2CASE(240);
        TOMO_F2CASE(256); TOMO_F2CASE(320);
#undef TOMO_F2CASE
        default: return false;
    }
}

// pass 1 of P = R * M for thread j2 < M: on entry v[j1] = x[j1 M + j2]; on exit v[k1] = Y[k1][j2].
// tw[t] = exp(-2 pi i t / P), t < P.
template <typename T, int R, int M, bool INV>
TOMO_HD void fft2_first(typename cx_of<T>::type *v, int j2, const typename cx_of<T>::type *__restrict__ tw) {
    typedef typename cx_of<T>::type C;
    SmallDft<T, R, INV>::run(v);
#pragma unroll
    for (int k1 = 1; k1 < R; ++k1) {
        const C w = tw[j2 * k1];
        v[k1] = INV ? cmulc(v[k1], w) : cmul(v[k1], w);
    }
}
// pass 2 for thread k1 < R: on entry v[j2] = Y[k1][j2]; on exit v[k2] = X[k1 + R k2].
template <typename T, int M, bool INV> TOMO_HD void fft2_second(typename cx_of<T>::type *v) { SmallDft<T, M, INV>::run(v); }

}  // namespace tomo
