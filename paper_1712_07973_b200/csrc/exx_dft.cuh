// exx_dft.cuh -- in-register complex fp64 DFT butterflies (radix 2,3,4 and composites 8,12,16) for sm_100a.
//
// Building block of the hand-written batched 3-D FFT that performs "Kernel 2" of PAPER.md:116,125-127
// (Poisson solve by FFT convolution).  All transforms here are the FORWARD transform
//     X[k] = sum_n x[n] exp(-2 pi i n k / R),   natural order in, natural order out, unnormalised.
// The inverse transform is obtained by calling the same routine with the real and imaginary arrays exchanged
// (IDFT(x) = swap(DFT(swap(x)))), which costs nothing in registers.
//
// Pruned variants for the Hockney zero padding ("appropriate padding"):
//   dft_ip<R>: inputs  x[R/2..R-1] are known to be zero (forward transform of a zero-padded line)
//   dft_op<R>: only outputs X[0..R/2-1] are produced   (inverse transform whose padded half is discarded)
//
// Twiddle constants are compile-time (multiples of 2 pi/48 cover R = 8, 12, 16); no runtime trigonometry,
// no recurrences (accuracy budget: SURVEY.md 8(c), 1e-11 parity needs table-quality twiddles).
#pragma once

#include <type_traits>

#ifndef EXX_HD
#define EXX_HD __host__ __device__ __forceinline__
#endif

namespace exx {

template <int I, int N, class F>
EXX_HD void static_for(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(static_cast<F&&>(f));
    }
}

// cos(2 pi j / 48), j = 0..12 (first quadrant), correctly rounded literals.
__host__ __device__ constexpr double cos48_q(int j) {
    constexpr double t[13] = {1.0,
                              0.99144486137381041114,
                              0.96592582628906828675,
                              0.92387953251128675613,
                              0.86602540378443864676,
                              0.79335334029123516458,
                              0.70710678118654752440,
                              0.60876142900872063942,
                              0.5,
                              0.38268343236508977173,
                              0.25881904510252076235,
                              0.13052619222005159155,
                              0.0};
    return t[j];
}
__host__ __device__ constexpr double cos48(int m) {
    m = ((m % 48) + 48) % 48;
    return m <= 12 ? cos48_q(m) : m <= 24 ? -cos48_q(24 - m) : m <= 36 ? -cos48_q(m - 24) : cos48_q(48 - m);
}
__host__ __device__ constexpr double sin48(int m) { return cos48(m - 12); }

// x *= W_R^M = exp(-2 pi i M / R)   (compile-time M, R | 48)
template <int R, int M>
EXX_HD void mul_w(double& xr, double& xi) {
    static_assert(48 % R == 0, "twiddle base must divide 48");
    constexpr int m = (((M % R) + R) % R) * (48 / R);      // in 48ths of a turn
    if constexpr (m == 0) {
    } else if constexpr (m == 12) {                         // * (-i)
        double t = xr; xr = xi; xi = -t;
    } else if constexpr (m == 24) {
        xr = -xr; xi = -xi;
    } else if constexpr (m == 36) {                         // * (+i)
        double t = xr; xr = -xi; xi = t;
    } else {
        constexpr double c = cos48(m), s = -sin48(m);       // W = c + i s
        double t = xr * c - xi * s;
        xi = xr * s + xi * c;
        xr = t;
    }
}

// ------------------------------------------------------------------------------------------------ bases
template <int R> struct Dft;     // full
template <int R> struct DftIP;   // inputs n >= R/2 are zero (values in the upper half are ignored)
template <int R> struct DftOP;   // outputs k <  R/2 only (upper half of the array is left unspecified)

template <> struct Dft<2> {
    EXX_HD static void run(double* xr, double* xi) {
        double ar = xr[0] + xr[1], ai = xi[0] + xi[1];
        xr[1] = xr[0] - xr[1]; xi[1] = xi[0] - xi[1];
        xr[0] = ar; xi[0] = ai;
    }
};
template <> struct DftIP<2> {
    EXX_HD static void run(double* xr, double* xi) { xr[1] = xr[0]; xi[1] = xi[0]; }
};
template <> struct DftOP<2> {
    EXX_HD static void run(double* xr, double* xi) { xr[0] += xr[1]; xi[0] += xi[1]; }
};

template <> struct Dft<3> {
    EXX_HD static void run(double* xr, double* xi) {
        constexpr double s = 0.86602540378443864676;        // sin(2 pi/3)
        double t1r = xr[1] + xr[2], t1i = xi[1] + xi[2];
        double t2r = xr[1] - xr[2], t2i = xi[1] - xi[2];
        double mr = xr[0] - 0.5 * t1r, mi = xi[0] - 0.5 * t1i;
        xr[0] += t1r; xi[0] += t1i;
        // X1 = m - i s t2 ; X2 = m + i s t2     (-i (a+ib) = b - ia)
        xr[1] = mr + s * t2i; xi[1] = mi - s * t2r;
        xr[2] = mr - s * t2i; xi[2] = mi + s * t2r;
    }
};

template <> struct Dft<4> {
    EXX_HD static void run(double* xr, double* xi) {
        double t0r = xr[0] + xr[2], t0i = xi[0] + xi[2];
        double t1r = xr[0] - xr[2], t1i = xi[0] - xi[2];
        double t2r = xr[1] + xr[3], t2i = xi[1] + xi[3];
        double t3r = xr[1] - xr[3], t3i = xi[1] - xi[3];
        xr[0] = t0r + t2r; xi[0] = t0i + t2i;
        xr[2] = t0r - t2r; xi[2] = t0i - t2i;
        xr[1] = t1r + t3i; xi[1] = t1i - t3r;               // t1 - i t3
        xr[3] = t1r - t3i; xi[3] = t1i + t3r;               // t1 + i t3
    }
};
template <> struct DftIP<4> {                               // x2 = x3 = 0
    EXX_HD static void run(double* xr, double* xi) {
        double ar = xr[0], ai = xi[0], br = xr[1], bi = xi[1];
        xr[0] = ar + br; xi[0] = ai + bi;
        xr[2] = ar - br; xi[2] = ai - bi;
        xr[1] = ar + bi; xi[1] = ai - br;
        xr[3] = ar - bi; xi[3] = ai + br;
    }
};
template <> struct DftOP<4> {                               // X0, X1 only
    EXX_HD static void run(double* xr, double* xi) {
        double t0r = xr[0] + xr[2], t0i = xi[0] + xi[2];
        double t1r = xr[0] - xr[2], t1i = xi[0] - xi[2];
        double t2r = xr[1] + xr[3], t2i = xi[1] + xi[3];
        double t3r = xr[1] - xr[3], t3i = xi[1] - xi[3];
        xr[0] = t0r + t2r; xi[0] = t0i + t2i;
        xr[1] = t1r + t3i; xi[1] = t1i - t3r;
    }
};

// ------------------------------------------------------------------------------------------------ composites
// Full:  n = Q n1 + n2, k = k1 + P k2.  Stage 1: P-point DFTs over n1, twiddle W_R^{n2 k1}; stage 2: Q-point over n2.
template <int R, int P, int Q, template <int> class First>
struct DftPQ {
    EXX_HD static void run(double* xr, double* xi) {
        static_assert(P * Q == R, "bad split");
        double yr[R], yi[R];
        static_for<0, Q>([&](auto N2) {
            constexpr int n2 = decltype(N2)::value;
            double ar[P], ai[P];
            static_for<0, P>([&](auto N1) { constexpr int n1 = decltype(N1)::value; ar[n1] = xr[Q * n1 + n2]; ai[n1] = xi[Q * n1 + n2]; });
            First<P>::run(ar, ai);
            static_for<0, P>([&](auto K1) {
                constexpr int k1 = decltype(K1)::value;
                mul_w<R, n2 * k1>(ar[k1], ai[k1]);
                yr[k1 * Q + n2] = ar[k1]; yi[k1 * Q + n2] = ai[k1];
            });
        });
        static_for<0, P>([&](auto K1) {
            constexpr int k1 = decltype(K1)::value;
            double br[Q], bi[Q];
            static_for<0, Q>([&](auto N2) { constexpr int n2 = decltype(N2)::value; br[n2] = yr[k1 * Q + n2]; bi[n2] = yi[k1 * Q + n2]; });
            Dft<Q>::run(br, bi);
            static_for<0, Q>([&](auto K2) { constexpr int k2 = decltype(K2)::value; xr[k1 + P * k2] = br[k2]; xi[k1 + P * k2] = bi[k2]; });
        });
    }
};

// Output-pruned: n = n1 + P n2, k = Q k1 + k2.  Stage 1: Q-point over n2, twiddle W_R^{n1 k2};
// stage 2: P-point over n1 keeping k1 < P/2  (k < R/2  <=>  k1 < P/2).
template <int R, int P, int Q>
struct DftPQ_OP {
    EXX_HD static void run(double* xr, double* xi) {
        static_assert(P * Q == R && P % 2 == 0, "bad split");
        double yr[R], yi[R];
        static_for<0, P>([&](auto N1) {
            constexpr int n1 = decltype(N1)::value;
            double br[Q], bi[Q];
            static_for<0, Q>([&](auto N2) { constexpr int n2 = decltype(N2)::value; br[n2] = xr[n1 + P * n2]; bi[n2] = xi[n1 + P * n2]; });
            Dft<Q>::run(br, bi);
            static_for<0, Q>([&](auto K2) {
                constexpr int k2 = decltype(K2)::value;
                mul_w<R, n1 * k2>(br[k2], bi[k2]);
                yr[k2 * P + n1] = br[k2]; yi[k2 * P + n1] = bi[k2];
            });
        });
        static_for<0, Q>([&](auto K2) {
            constexpr int k2 = decltype(K2)::value;
            double ar[P], ai[P];
            static_for<0, P>([&](auto N1) { constexpr int n1 = decltype(N1)::value; ar[n1] = yr[k2 * P + n1]; ai[n1] = yi[k2 * P + n1]; });
            DftOP<P>::run(ar, ai);
            static_for<0, P / 2>([&](auto K1) { constexpr int k1 = decltype(K1)::value; xr[Q * k1 + k2] = ar[k1]; xi[Q * k1 + k2] = ai[k1]; });
        });
    }
};

template <> struct Dft<6>    { EXX_HD static void run(double* r, double* i) { DftPQ<6, 2, 3, Dft>::run(r, i); } };
template <> struct DftIP<6>  { EXX_HD static void run(double* r, double* i) { DftPQ<6, 2, 3, DftIP>::run(r, i); } };
template <> struct DftOP<6>  { EXX_HD static void run(double* r, double* i) { DftPQ_OP<6, 2, 3>::run(r, i); } };
template <> struct Dft<8>    { EXX_HD static void run(double* r, double* i) { DftPQ<8, 4, 2, Dft>::run(r, i); } };
template <> struct Dft<12>   { EXX_HD static void run(double* r, double* i) { DftPQ<12, 4, 3, Dft>::run(r, i); } };
template <> struct Dft<16>   { EXX_HD static void run(double* r, double* i) { DftPQ<16, 4, 4, Dft>::run(r, i); } };
template <> struct DftIP<8>  { EXX_HD static void run(double* r, double* i) { DftPQ<8, 4, 2, DftIP>::run(r, i); } };
template <> struct DftIP<12> { EXX_HD static void run(double* r, double* i) { DftPQ<12, 4, 3, DftIP>::run(r, i); } };
template <> struct DftIP<16> { EXX_HD static void run(double* r, double* i) { DftPQ<16, 4, 4, DftIP>::run(r, i); } };
template <> struct DftOP<8>  { EXX_HD static void run(double* r, double* i) { DftPQ_OP<8, 4, 2>::run(r, i); } };
template <> struct DftOP<12> { EXX_HD static void run(double* r, double* i) { DftPQ_OP<12, 4, 3>::run(r, i); } };
template <> struct DftOP<16> { EXX_HD static void run(double* r, double* i) { DftPQ_OP<16, 4, 4>::run(r, i); } };

// Direction / pruning selectors used by the pass kernels.
//   fwd<R, PRUNED>: forward DFT, inputs >= R/2 zero if PRUNED.      inv<R, PRUNED>: inverse DFT, outputs < R/2 only if PRUNED.
template <int R, bool PRUNED>
EXX_HD void dft_fwd(double* xr, double* xi) {
    if constexpr (PRUNED) DftIP<R>::run(xr, xi); else Dft<R>::run(xr, xi);
}
template <int R, bool PRUNED>
EXX_HD void dft_inv(double* xr, double* xi) {
    if constexpr (PRUNED) DftOP<R>::run(xi, xr); else Dft<R>::run(xi, xr);
}

}  // namespace exx
