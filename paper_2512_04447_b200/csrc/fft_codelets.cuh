// Register-resident forward DFT codelets (e^{-2 pi i nk/R}), separate re[]/im[] arrays so
// that the inverse transform is the SAME code called with (im, re): swap . F . swap = R * F^-1.
// Part of the CUDA path of librsdft (PAPER.md:19 task (1), "FFT used to apply the Laplacian").
// Constants are literals rounded from 40-digit values; nothing here is shared with oracle/.
#pragma once
#include <type_traits>

namespace rsdft {

template <int I, int N, class F>
__device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// cos(2 pi m / R), sin(2 pi m / R) for the radices the codelets use internally.
template <int R> struct Trig;
template <> struct Trig<1> { static constexpr double c[1] = {1.0}; static constexpr double s[1] = {0.0}; };
template <> struct Trig<2> { static constexpr double c[2] = {1.0, -1.0}; static constexpr double s[2] = {0.0, 0.0}; };
template <> struct Trig<3> {
    static constexpr double c[3] = {1.0, -0.5, -0.5};
    static constexpr double s[3] = {0.0, 0.866025403784438646764, -0.866025403784438646764};
};
template <> struct Trig<4> { static constexpr double c[4] = {1.0, 0.0, -1.0, 0.0}; static constexpr double s[4] = {0.0, 1.0, 0.0, -1.0}; };
template <> struct Trig<5> {
    static constexpr double c[5] = {1.0, 0.309016994374947424102, -0.809016994374947424102,
                                    -0.809016994374947424102, 0.309016994374947424102};
    static constexpr double s[5] = {0.0, 0.951056516295153572116, 0.587785252292473129169,
                                    -0.587785252292473129169, -0.951056516295153572116};
};
template <> struct Trig<6> {
    static constexpr double c[6] = {1.0, 0.5, -0.5, -1.0, -0.5, 0.5};
    static constexpr double s[6] = {0.0, 0.866025403784438646764, 0.866025403784438646764, 0.0,
                                    -0.866025403784438646764, -0.866025403784438646764};
};
template <> struct Trig<7> {
    static constexpr double c[7] = {1.0, 0.623489801858733530525, -0.222520933956314404289,
                                    -0.900968867902419126236, -0.900968867902419126236,
                                    -0.222520933956314404289, 0.623489801858733530525};
    static constexpr double s[7] = {0.0, 0.781831482468029808708, 0.974927912181823607018,
                                    0.433883739117558120476, -0.433883739117558120476,
                                    -0.974927912181823607018, -0.781831482468029808708};
};
template <> struct Trig<8> {
    static constexpr double c[8] = {1.0, 0.707106781186547524401, 0.0, -0.707106781186547524401,
                                    -1.0, -0.707106781186547524401, 0.0, 0.707106781186547524401};
    static constexpr double s[8] = {0.0, 0.707106781186547524401, 1.0, 0.707106781186547524401,
                                    0.0, -0.707106781186547524401, -1.0, -0.707106781186547524401};
};
template <> struct Trig<10> {
    static constexpr double c[10] = {1.00000000000000000000, 0.809016994374947424102, 0.309016994374947424102, -0.309016994374947424102, -0.809016994374947424102, -1.00000000000000000000, -0.809016994374947424102, -0.309016994374947424102, 0.309016994374947424102, 0.809016994374947424102};
    static constexpr double s[10] = {0.0, 0.587785252292473129169, 0.951056516295153572116, 0.951056516295153572116, 0.587785252292473129169, 0.0, -0.587785252292473129169, -0.951056516295153572116, -0.951056516295153572116, -0.587785252292473129169};
};
template <> struct Trig<12> {
    static constexpr double c[12] = {1.00000000000000000000, 0.866025403784438646764, 0.500000000000000000000, 0.0, -0.500000000000000000000, -0.866025403784438646764, -1.00000000000000000000, -0.866025403784438646764, -0.500000000000000000000, 0.0, 0.500000000000000000000, 0.866025403784438646764};
    static constexpr double s[12] = {0.0, 0.500000000000000000000, 0.866025403784438646764, 1.00000000000000000000, 0.866025403784438646764, 0.500000000000000000000, 0.0, -0.500000000000000000000, -0.866025403784438646764, -1.00000000000000000000, -0.866025403784438646764, -0.500000000000000000000};
};
template <> struct Trig<16> {
    static constexpr double c[16] = {1.0, 0.923879532511286756128, 0.707106781186547524401, 0.382683432365089771728,
                                     0.0, -0.382683432365089771728, -0.707106781186547524401, -0.923879532511286756128,
                                     -1.0, -0.923879532511286756128, -0.707106781186547524401, -0.382683432365089771728,
                                     0.0, 0.382683432365089771728, 0.707106781186547524401, 0.923879532511286756128};
    static constexpr double s[16] = {0.0, 0.382683432365089771728, 0.707106781186547524401, 0.923879532511286756128,
                                     1.0, 0.923879532511286756128, 0.707106781186547524401, 0.382683432365089771728,
                                     0.0, -0.382683432365089771728, -0.707106781186547524401, -0.923879532511286756128,
                                     -1.0, -0.923879532511286756128, -0.707106781186547524401, -0.382683432365089771728};
};

// (re, im) *= (c - i s)   [general forward twiddle, 2 mul + 2 fma]
__device__ __forceinline__ void tw_mul(double &re, double &im, double c, double s)
{
    const double r = re, i = im;
    re = fma(i, s, r * c);
    im = fma(-r, s, i * c);
}

// (re, im) *= e^{-2 pi i m / R}, m and R compile-time; multiples of 1/8 turn are special-cased.
template <int R, int MM>
__device__ __forceinline__ void tw_mul_const(double &re, double &im)
{
    constexpr int m = ((MM % R) + R) % R;
    if constexpr (m == 0) {
    } else if constexpr (4 * m == R) {          // -i
        const double r = re; re = im; im = -r;
    } else if constexpr (2 * m == R) {          // -1
        re = -re; im = -im;
    } else if constexpr (4 * m == 3 * R) {      // +i
        const double r = re; re = -im; im = r;
    } else if constexpr (8 * m == R) {          // (1 - i)/sqrt2
        const double r = re, i = im, h = 0.707106781186547524401;
        re = (r + i) * h; im = (i - r) * h;
    } else if constexpr (8 * m == 3 * R) {      // (-1 - i)/sqrt2
        const double r = re, i = im, h = 0.707106781186547524401;
        re = (i - r) * h; im = -(r + i) * h;
    } else if constexpr (8 * m == 5 * R) {      // (-1 + i)/sqrt2
        const double r = re, i = im, h = 0.707106781186547524401;
        re = -(r + i) * h; im = (r - i) * h;
    } else if constexpr (8 * m == 7 * R) {      // (1 + i)/sqrt2
        const double r = re, i = im, h = 0.707106781186547524401;
        re = (r - i) * h; im = (r + i) * h;
    } else {
        constexpr double cc = Trig<R>::c[m], ss = Trig<R>::s[m];
        tw_mul(re, im, cc, ss);
    }
}

template <int R> struct Dft;

template <> struct Dft<1> {
    static __device__ __forceinline__ void run(double (&)[1], double (&)[1]) {}
};

template <> struct Dft<2> {
    static __device__ __forceinline__ void run(double (&re)[2], double (&im)[2])
    {
        const double r0 = re[0], i0 = im[0];
        re[0] = r0 + re[1]; im[0] = i0 + im[1];
        re[1] = r0 - re[1]; im[1] = i0 - im[1];
    }
};

template <> struct Dft<4> {
    static __device__ __forceinline__ void run(double (&re)[4], double (&im)[4])
    {
        const double t0r = re[0] + re[2], t0i = im[0] + im[2];
        const double t1r = re[0] - re[2], t1i = im[0] - im[2];
        const double t2r = re[1] + re[3], t2i = im[1] + im[3];
        const double t3r = re[1] - re[3], t3i = im[1] - im[3];
        re[0] = t0r + t2r; im[0] = t0i + t2i;
        re[2] = t0r - t2r; im[2] = t0i - t2i;
        re[1] = t1r + t3i; im[1] = t1i - t3r;   // t1 - i t3
        re[3] = t1r - t3i; im[3] = t1i + t3r;   // t1 + i t3
    }
};

// Odd prime P: pair sums/differences, X_k = A_k - i B_k, X_{P-k} = A_k + i B_k.
template <int P>
struct DftPrime {
    static __device__ __forceinline__ void run(double (&re)[P], double (&im)[P])
    {
        constexpr int H = (P - 1) / 2;
        double sr[H], si[H], dr[H], di[H];
#pragma unroll
        for (int j = 0; j < H; ++j) {
            sr[j] = re[j + 1] + re[P - 1 - j]; si[j] = im[j + 1] + im[P - 1 - j];
            dr[j] = re[j + 1] - re[P - 1 - j]; di[j] = im[j + 1] - im[P - 1 - j];
        }
        const double a0r = re[0], a0i = im[0];
        double x0r = a0r, x0i = a0i;
#pragma unroll
        for (int j = 0; j < H; ++j) { x0r += sr[j]; x0i += si[j]; }
        re[0] = x0r; im[0] = x0i;
        static_for<1, H + 1>([&](auto K) {
            constexpr int k = decltype(K)::value;
            double ar = a0r, ai = a0i, br = 0.0, bi = 0.0;
            static_for<1, H + 1>([&](auto J) {
                constexpr int j = decltype(J)::value;
                constexpr int idx = (j * k) % P;
                constexpr double cc = Trig<P>::c[idx], ss = Trig<P>::s[idx];
                ar = fma(cc, sr[j - 1], ar);
                ai = fma(cc, si[j - 1], ai);
                if constexpr (j == 1) { br = ss * dr[0]; bi = ss * di[0]; }
                else { br = fma(ss, dr[j - 1], br); bi = fma(ss, di[j - 1], bi); }
            });
            re[k] = ar + bi;     im[k] = ai - br;
            re[P - k] = ar - bi; im[P - k] = ai + br;
        });
    }
};
template <> struct Dft<3> : DftPrime<3> {};
template <> struct Dft<5> : DftPrime<5> {};
template <> struct Dft<7> : DftPrime<7> {};

// Cooley-Tukey R = R1*R2 in registers: n = n1*R2 + n2, k = k1 + R1*k2.
template <int R1, int R2>
struct DftCT {
    static constexpr int R = R1 * R2;
    static __device__ __forceinline__ void run(double (&re)[R], double (&im)[R])
    {
        double yr[R], yi[R];       // y[k1*R2 + n2]
        static_for<0, R2>([&](auto N2) {
            constexpr int n2 = decltype(N2)::value;
            double ar[R1], ai[R1];
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) { ar[n1] = re[n1 * R2 + n2]; ai[n1] = im[n1 * R2 + n2]; }
            Dft<R1>::run(ar, ai);
            static_for<0, R1>([&](auto K1) {
                constexpr int k1 = decltype(K1)::value;
                tw_mul_const<R, n2 * k1>(ar[k1], ai[k1]);
                yr[k1 * R2 + n2] = ar[k1]; yi[k1 * R2 + n2] = ai[k1];
            });
        });
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) {
            double br[R2], bi[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) { br[n2] = yr[k1 * R2 + n2]; bi[n2] = yi[k1 * R2 + n2]; }
            Dft<R2>::run(br, bi);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) { re[k1 + R1 * k2] = br[k2]; im[k1 + R1 * k2] = bi[k2]; }
        }
    }
};
template <> struct Dft<6> : DftCT<2, 3> {};
template <> struct Dft<8> : DftCT<2, 4> {};
template <> struct Dft<10> : DftCT<2, 5> {};
template <> struct Dft<12> : DftCT<3, 4> {};
template <> struct Dft<16> : DftCT<4, 4> {};

}  // namespace rsdft
