// CPU harness for csrc/fft_device.cuh: the same template code the kernels use, compiled by g++ with one lane,
// checked against a direct O(P^2) DFT in fp64.  Prints "P <fwd32> <inv32> <fwd64> <inv64>" per size.
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "fft_device.cuh"
#include "fft_reg.cuh"
using namespace tomo;

static void plan(int P, FftDesc &d) {
    d.P = P; d.nrad = 0;
    int r = P;
    while (r % 5 == 0) { d.rad[d.nrad++] = 5; r /= 5; }
    while (r % 3 == 0) { d.rad[d.nrad++] = 3; r /= 3; }
    while (r % 8 == 0) { d.rad[d.nrad++] = 8; r /= 8; }
    while (r % 4 == 0) { d.rad[d.nrad++] = 4; r /= 4; }
    while (r % 2 == 0) { d.rad[d.nrad++] = 2; r /= 2; }
}

template <typename T> static double run(int P, bool inv) {
    typedef typename cx_of<T>::type C;
    FftDesc d;
    plan(P, d);
    std::vector<C> a(P), b(P), tw(P);
    std::vector<std::complex<double>> in(P);
    for (int i = 0; i < P; ++i) {
        in[i] = {std::sin(i * 1.3) + 0.01 * i, std::cos(i * 0.7) - 0.3};
        a[i].x = (T)in[i].real(); a[i].y = (T)in[i].imag();
        tw[i].x = (T)std::cos(2 * M_PI * i / P); tw[i].y = (T)-std::sin(2 * M_PI * i / P);
    }
    C *r = inv ? warp_fft<T, true, 1>(a.data(), b.data(), d, tw.data(), 0) : warp_fft<T, false, 1>(a.data(), b.data(), d, tw.data(), 0);
    double err = 0, nrm = 0;
    for (int k = 0; k < P; ++k) {
        std::complex<double> s = 0;
        for (int j = 0; j < P; ++j) {
            const double ph = (inv ? 1 : -1) * 2 * M_PI * (double)(((long)j * k) % P) / P;
            s += in[j] * std::complex<double>(std::cos(ph), std::sin(ph));
        }
        err += std::norm(s - std::complex<double>(r[k].x, r[k].y));
        nrm += std::norm(s);
    }
    return std::sqrt(err / nrm);
}

// the compile-time-planned chain (warp_fft_static) for the sizes the persistent kernel instantiates
template <typename T, int P> static double run_static(bool inv) {
    typedef typename cx_of<T>::type C;
    std::vector<C> a(P), b(P), tw(P);
    std::vector<std::complex<double>> in(P);
    for (int i = 0; i < P; ++i) {
        in[i] = {std::sin(i * 1.3) + 0.01 * i, std::cos(i * 0.7) - 0.3};
        a[i].x = (T)in[i].real(); a[i].y = (T)in[i].imag();
        tw[i].x = (T)std::cos(2 * M_PI * i / P); tw[i].y = (T)-std::sin(2 * M_PI * i / P);
    }
    C *r = inv ? warp_fft_static<T, true, P, 1>(a.data(), b.data(), tw.data(), 0) : warp_fft_static<T, false, P, 1>(a.data(), b.data(), tw.data(), 0);
    // same result buffer as the run-time plan: first argument iff the number of passes is even
    if ((r == a.data()) != (CountPasses<P>::value % 2 == 0)) return 1.0;
    double err = 0, nrm = 0;
    for (int k = 0; k < P; ++k) {
        std::complex<double> s = 0;
        for (int j = 0; j < P; ++j) {
            const double ph = (inv ? 1 : -1) * 2 * M_PI * (double)(((long)j * k) % P) / P;
            s += in[j] * std::complex<double>(std::cos(ph), std::sin(ph));
        }
        err += std::norm(s - std::complex<double>(r[k].x, r[k].y));
        nrm += std::norm(s);
    }
    return std::sqrt(err / nrm);
}
template <int P> static void print_static() {
    std::printf("S %d %.3e %.3e %.3e %.3e\n", P, run_static<float, P>(false), run_static<float, P>(true), run_static<double, P>(false),
                run_static<double, P>(true));
}

// the register two-pass split (fft_reg.cuh) used by the persistent kernel: threads emulated one after the other,
// both orders of the split (R = A, M = B and R = B, M = A), padded intermediate layout as on the device
template <typename T, int P, int R, int M> static double run_reg(bool inv) {
    typedef typename cx_of<T>::type C;
    std::vector<C> tw(P), Y((size_t)R * (M + 1)), out(P);
    std::vector<std::complex<double>> in(P);
    for (int i = 0; i < P; ++i) {
        in[i] = {std::sin(i * 1.3) + 0.01 * i, std::cos(i * 0.7) - 0.3};
        tw[i].x = (T)std::cos(2 * M_PI * i / P); tw[i].y = (T)-std::sin(2 * M_PI * i / P);
    }
    for (int j2 = 0; j2 < M; ++j2) {
        C v[R];
        for (int j1 = 0; j1 < R; ++j1) { v[j1].x = (T)in[j1 * M + j2].real(); v[j1].y = (T)in[j1 * M + j2].imag(); }
        if (inv) fft2_first<T, R, M, true>(v, j2, tw.data()); else fft2_first<T, R, M, false>(v, j2, tw.data());
        for (int k1 = 0; k1 < R; ++k1) Y[(size_t)k1 * (M + 1) + j2] = v[k1];
    }
    for (int k1 = 0; k1 < R; ++k1) {
        C v[M];
        for (int j2 = 0; j2 < M; ++j2) v[j2] = Y[(size_t)k1 * (M + 1) + j2];
        if (inv) fft2_second<T, M, true>(v); else fft2_second<T, M, false>(v);
        for (int k2 = 0; k2 < M; ++k2) out[k1 + R * k2] = v[k2];
    }
    double err = 0, nrm = 0;
    for (int k = 0; k < P; ++k) {
        std::complex<double> s = 0;
        for (int j = 0; j < P; ++j) {
            const double ph = (inv ? 1 : -1) * 2 * M_PI * (double)(((long)j * k) % P) / P;
            s += in[j] * std::complex<double>(std::cos(ph), std::sin(ph));
        }
        err += std::norm(s - std::complex<double>(out[k].x, out[k].y));
        nrm += std::norm(s);
    }
    return std::sqrt(err / nrm);
}
template <int P> static void print_reg() {
    constexpr int A = Fact2<P>::A, B = Fact2<P>::B;
    static_assert(A * B == P, "Fact2");
    std::printf("R %d %.3e %.3e %.3e %.3e %.3e %.3e %.3e %.3e\n", P, run_reg<float, P, A, B>(false), run_reg<float, P, A, B>(true),
                run_reg<double, P, A, B>(false), run_reg<double, P, A, B>(true), run_reg<float, P, B, A>(false),
                run_reg<float, P, B, A>(true), run_reg<double, P, B, A>(false), run_reg<double, P, B, A>(true));
}

int main(int argc, char **argv) {
    if (argc > 1 && argv[1][0] == 'R') {
        print_reg<16>(); print_reg<20>(); print_reg<24>(); print_reg<32>(); print_reg<40>(); print_reg<48>(); print_reg<64>();
        print_reg<80>(); print_reg<128>(); print_reg<160>(); print_reg<180>(); print_reg<192>(); print_reg<240>(); print_reg<256>();
        print_reg<320>();
        return 0;
    }
    if (argc > 1 && argv[1][0] == 'S') {
        print_static<16>(); print_static<20>(); print_static<24>(); print_static<32>(); print_static<40>(); print_static<48>();
        print_static<64>(); print_static<80>(); print_static<128>(); print_static<160>(); print_static<180>(); print_static<192>();
        print_static<240>(); print_static<256>(); print_static<320>();
        return 0;
    }
    for (int i = 1; i < argc; ++i) {
        const int P = std::atoi(argv[i]);
        std::printf("%d %.3e %.3e %.3e %.3e\n", P, run<float>(P, false), run<float>(P, true), run<double>(P, false), run<double>(P, true));
    }
    return 0;
}
