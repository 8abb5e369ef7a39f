// sht_dft_codelets.cuh -- R-point DFTs in registers for the mixed-radix ring transforms (sht_ring_mixed.cu):
// any R whose prime factors are <= 31, natural order in and out, forward (e^{-2 pi i n k / R}) or inverse (e^{+...}).
//   prime R      : direct sums over the pairs x_j +- x_{R-j} (R^2 / 2 real multiply-adds per output pair)
//   composite R  : Cooley-Tukey R = A B (A the smallest prime factor): B-point transforms over n1 (n = B... see below),
//                  compile-time twiddles, A-point transforms -- all indices resolved at compile time
// The trigonometric constants are evaluated at compile time (constexpr series in long double, argument reduced to
// [0, pi/4]), so no table is read at run time.
#pragma once
#include <cuda_runtime.h>

namespace sht {
namespace dftc {

#define SHT_HD __host__ __device__ __forceinline__

constexpr long double PI_L = 3.14159265358979323846264338327950288419716939937510L;

// sin / cos of x in [0, pi/4] by their Taylor series (20 terms: far below 1e-19)
__host__ __device__ constexpr long double sin_small(long double x)
{
    long double term = x, sum = x;
    for (int k = 1; k < 20; ++k) { term *= -x * x / ((2 * k) * (2 * k + 1)); sum += term; }
    return sum;
}
__host__ __device__ constexpr long double cos_small(long double x)
{
    long double term = 1.0L, sum = 1.0L;
    for (int k = 1; k < 20; ++k) { term *= -x * x / ((2 * k - 1) * (2 * k)); sum += term; }
    return sum;
}
// cos(2 pi k / R), sin(2 pi k / R) with the argument reduced exactly in integers (eighths of the circle)
__host__ __device__ constexpr long double cos2pi(long long k, long long R)
{
    k %= R; if (k < 0) k += R;
    // angle = 2 pi k / R; reduce to the first octant using 8 k / R
    if (2 * k > R) return cos2pi(R - k, R);                       // cos(2 pi - a) = cos a
    if (4 * k > R) return -cos2pi(R - 2 * k, 2 * R);              // cos(pi - a) = -cos a, a = 2 pi (R - 2k) / (2R)
    if (8 * k > R) return sin_small(2.0L * PI_L * (long double)(R - 4 * k) / (long double)(4 * R));   // cos(pi/2 - a) = sin a
    return cos_small(2.0L * PI_L * (long double)k / (long double)R);
}
__host__ __device__ constexpr long double sin2pi(long long k, long long R)
{
    k %= R; if (k < 0) k += R;
    if (2 * k > R) return -sin2pi(R - k, R);
    if (4 * k > R) return sin2pi(R - 2 * k, 2 * R);               // sin(pi - a) = sin a
    if (8 * k > R) return cos_small(2.0L * PI_L * (long double)(R - 4 * k) / (long double)(4 * R));   // sin(pi/2 - a) = cos a
    return sin_small(2.0L * PI_L * (long double)k / (long double)R);
}

__host__ __device__ constexpr int smallest_factor(int r)
{
    for (int f = 2; f * f <= r; ++f) if (r % f == 0) return f;
    return r;
}

SHT_HD double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
SHT_HD double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }

// a * exp(-+ 2 pi i K / R) (- forward, + if INV), K and R compile-time; trivial multiples of a quarter turn are free
template <int K, int R, bool INV>
SHT_HD double2 mul_root(double2 a)
{
    constexpr int k = ((K % R) + R) % R;
    if constexpr (k == 0) return a;
    else if constexpr (4 * k == R) return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
    else if constexpr (2 * k == R) return make_double2(-a.x, -a.y);
    else if constexpr (4 * k == 3 * R) return INV ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);
    else {
        constexpr double c = (double)cos2pi(k, R);
        constexpr double s = (double)(INV ? sin2pi(k, R) : -sin2pi(k, R));       // imaginary part of the root
        return make_double2(fma(a.x, c, -(a.y * s)), fma(a.x, s, a.y * c));
    }
}

template <int R, bool INV> struct Dft;

// prime radix: x_0 + sum_j cos(2 pi j s / R)(x_j + x_{R-j}) -+ i sum_j sin(2 pi j s / R)(x_j - x_{R-j})
template <int R, bool INV>
struct DftPrime {
    template <int S, int J>
    static SHT_HD void acc(const double2* a, const double2* b, double2& re, double2& im)
    {
        if constexpr (J <= (R - 1) / 2) {
            constexpr double c = (double)cos2pi((long long)J * S, R), s = (double)sin2pi((long long)J * S, R);
            re.x = fma(c, a[J - 1].x, re.x); re.y = fma(c, a[J - 1].y, re.y);
            im.x = fma(s, b[J - 1].x, im.x); im.y = fma(s, b[J - 1].y, im.y);
            acc<S, J + 1>(a, b, re, im);
        }
    }
    template <int S>
    static SHT_HD void outs(const double2* a, const double2* b, double2 x0, double2* u)
    {
        if constexpr (S <= (R - 1) / 2) {
            double2 re = x0, im = make_double2(0.0, 0.0);
            acc<S, 1>(a, b, re, im);
            // forward: X_s = re - i im, X_{R-s} = re + i im; inverse: the other way round
            const double2 lo = make_double2(re.x + im.y, re.y - im.x), hi = make_double2(re.x - im.y, re.y + im.x);
            u[S] = INV ? hi : lo;
            u[R - S] = INV ? lo : hi;
            outs<S + 1>(a, b, x0, u);
        }
    }
    static SHT_HD void run(double2* u)
    {
        if constexpr (R == 2) {
            const double2 a = u[0], b = u[1];
            u[0] = cadd(a, b); u[1] = csub(a, b);
        } else {
            constexpr int H = (R - 1) / 2;
            double2 a[H], b[H];
            const double2 x0 = u[0];
            double2 sum = x0;
#pragma unroll
            for (int j = 1; j <= H; ++j) { a[j - 1] = cadd(u[j], u[R - j]); b[j - 1] = csub(u[j], u[R - j]); sum = cadd(sum, a[j - 1]); }
            u[0] = sum;
            outs<1>(a, b, x0, u);
        }
    }
};

// composite radix R = A B: n = B n1 + n2 (n1 < A, n2 < B), k = k1 + A k2 (k1 < A, k2 < B):
//   X[k1 + A k2] = sum_n2 w_B^{n2 k2} { w_R^{n2 k1} sum_n1 x[B n1 + n2] w_A^{n1 k1} }
template <int R, int A, bool INV>
struct DftCT {
    static constexpr int B = R / A;
    template <int N2, int K1>
    static SHT_HD void twiddle_row(double2 (*t)[A])
    {
        if constexpr (K1 < A) {
            t[N2][K1] = mul_root<N2 * K1, R, INV>(t[N2][K1]);
            twiddle_row<N2, K1 + 1>(t);
        }
    }
    template <int N2>
    static SHT_HD void inner(const double2* u, double2 (*t)[A])
    {
        if constexpr (N2 < B) {
#pragma unroll
            for (int n1 = 0; n1 < A; ++n1) t[N2][n1] = u[B * n1 + N2];
            Dft<A, INV>::run(t[N2]);
            twiddle_row<N2, 1>(t);
            inner<N2 + 1>(u, t);
        }
    }
    static SHT_HD void run(double2* u)
    {
        double2 t[B][A];
        inner<0>(u, t);
#pragma unroll
        for (int k1 = 0; k1 < A; ++k1) {
            double2 v[B];
#pragma unroll
            for (int n2 = 0; n2 < B; ++n2) v[n2] = t[n2][k1];
            Dft<B, INV>::run(v);
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) u[k1 + A * k2] = v[k2];
        }
    }
};

template <int R, bool INV>
struct Dft {
    static SHT_HD void run(double2* u)
    {
        if constexpr (R == 1) { }
        else if constexpr (R == 4) {
            // radix 4 directly (no multiplications)
            const double2 v0 = cadd(u[0], u[2]), v1 = csub(u[0], u[2]), v2 = cadd(u[1], u[3]), dd = csub(u[1], u[3]);
            const double2 v3 = INV ? make_double2(-dd.y, dd.x) : make_double2(dd.y, -dd.x);
            u[0] = cadd(v0, v2); u[1] = cadd(v1, v3); u[2] = csub(v0, v2); u[3] = csub(v1, v3);
        }
        else if constexpr (smallest_factor(R) == R) DftPrime<R, INV>::run(u);
        else if constexpr (R % 4 == 0 && R > 4) DftCT<R, 4, INV>::run(u);
        else DftCT<R, smallest_factor(R), INV>::run(u);
    }
};

// u[k] *= w^k, k = 1 .. R-1 (any R >= 2): w, w^2, w^3 and the running (w^4)^i
template <int R>
SHT_HD void mul_powers_any(double2* u, double2 w)
{
    auto cm = [](double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); };
    if constexpr (R >= 2) u[1] = cm(u[1], w);
    if constexpr (R >= 3) {
        const double2 w2 = cm(w, w);
        u[2] = cm(u[2], w2);
        if constexpr (R >= 4) {
            const double2 w3 = cm(w2, w), w4 = cm(w2, w2);
            u[3] = cm(u[3], w3);
            double2 b = w4;
#pragma unroll
            for (int i = 1; 4 * i < R; ++i) {
                u[4 * i] = cm(u[4 * i], b);
                if (4 * i + 1 < R) u[4 * i + 1] = cm(u[4 * i + 1], cm(b, w));
                if (4 * i + 2 < R) u[4 * i + 2] = cm(u[4 * i + 2], cm(b, w2));
                if (4 * i + 3 < R) u[4 * i + 3] = cm(u[4 * i + 3], cm(b, w3));
                if (4 * (i + 1) < R) b = cm(b, w4);
            }
        }
    }
}

#undef SHT_HD

}  // namespace dftc
}  // namespace sht
