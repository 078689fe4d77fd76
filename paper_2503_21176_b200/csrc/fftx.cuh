// fftx.cuh -- small complex DFTs held entirely in registers (sizes 2..16 with factors 2, 3, 5), the building block of
// the two-step x-axis transform in fftx.cu.  Every index below is a compile-time constant (static_for over
// std::integral_constant), so the arrays live in registers and the twiddle factors are immediates.
// Not an algorithm of the paper: a-5/a-7 (Alg. 2 steps 2 and 4, "FFT") are library calls there.
#pragma once
#include <cuda_runtime.h>
#include <type_traits>

namespace fx {

#define FX_HD __host__ __device__ __forceinline__

template <int I, int E, class F>
FX_HD void sfor(F&& f)
{
    if constexpr (I < E) {
        f(std::integral_constant<int, I>{});
        sfor<I + 1, E>(f);
    }
}

// compile-time cos/sin of 2 pi k / n (Taylor series about 0 after folding the angle into (-pi, pi]; 20 terms: below
// 1e-16 absolute, far under fp32 rounding)
constexpr double fx_pi = 3.14159265358979323846264338327950288;
__host__ __device__ constexpr double fx_angle(int k, int n)
{
    k %= n;
    if (k < 0) k += n;
    if (2 * k > n) k -= n;
    return 2.0 * fx_pi * (double)k / (double)n;
}
__host__ __device__ constexpr double fx_cos(int k, int n)
{
    const double x = fx_angle(k, n), x2 = x * x;
    double term = 1.0, sum = 1.0;
    for (int j = 1; j <= 20; ++j) {
        term *= -x2 / (double)((2 * j - 1) * (2 * j));
        sum += term;
    }
    return sum;
}
__host__ __device__ constexpr double fx_sin(int k, int n)
{
    const double x = fx_angle(k, n), x2 = x * x;
    double term = x, sum = x;
    for (int j = 1; j <= 20; ++j) {
        term *= -x2 / (double)((2 * j) * (2 * j + 1));
        sum += term;
    }
    return sum;
}

FX_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
FX_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
FX_HD float2 cmulf(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// a * e^{-+ 2 pi i K / N}  (forward: minus; INV: plus), K and N compile-time
template <int K, int N, bool INV>
FX_HD float2 twmul(float2 a)
{
    constexpr int k = ((K % N) + N) % N;
    if constexpr (k == 0) return a;
    else if constexpr (2 * k == N) return make_float2(-a.x, -a.y);
    else if constexpr (4 * k == N) return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);          // * (+-i)
    else if constexpr (4 * k == 3 * N) return INV ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
    else {
        constexpr float c = (float)fx_cos(k, N);
        constexpr float s = (float)(INV ? fx_sin(k, N) : -fx_sin(k, N));
        return make_float2(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}

template <int N>
__host__ __device__ constexpr int first_factor()
{
    if (N > 4 && N % 4 == 0) return 4;
    if (N % 2 == 0) return 2;
    if (N % 3 == 0) return 3;
    if (N % 5 == 0) return 5;
    return N;
}

// In-place DFT of v[0..N): v[k] <- sum_n v[n] e^{-+ 2 pi i n k / N}, natural order in and out.
template <int N, bool INV>
struct Dft {
    static FX_HD void run(float2 (&v)[N])
    {
        constexpr int A = first_factor<N>(), B = N / A;
        static_assert(A < N, "unsupported prime size");
        float2 t[N];                                        // t[ka * B + b]
        sfor<0, B>([&](auto b_) {
            constexpr int b = decltype(b_)::value;
            float2 u[A];
            sfor<0, A>([&](auto a_) { constexpr int a = decltype(a_)::value; u[a] = v[B * a + b]; });
            Dft<A, INV>::run(u);
            sfor<0, A>([&](auto k_) { constexpr int ka = decltype(k_)::value; t[ka * B + b] = twmul<ka * b, N, INV>(u[ka]); });
        });
        sfor<0, A>([&](auto k_) {
            constexpr int ka = decltype(k_)::value;
            float2 u[B];
            sfor<0, B>([&](auto b_) { constexpr int b = decltype(b_)::value; u[b] = t[ka * B + b]; });
            Dft<B, INV>::run(u);
            sfor<0, B>([&](auto q_) { constexpr int kb = decltype(q_)::value; v[ka + A * kb] = u[kb]; });
        });
    }
};

template <bool INV> struct Dft<1, INV> { static FX_HD void run(float2 (&)[1]) {} };

template <bool INV>
struct Dft<2, INV> {
    static FX_HD void run(float2 (&v)[2])
    {
        const float2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};

template <bool INV>
struct Dft<4, INV> {
    static FX_HD void run(float2 (&v)[4])
    {
        const float2 a = cadd(v[0], v[2]), b = csub(v[0], v[2]), c = cadd(v[1], v[3]), d = csub(v[1], v[3]);
        const float2 id = INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);       // (+-i) d, forward: -i d
        v[0] = cadd(a, c);
        v[2] = csub(a, c);
        v[1] = cadd(b, id);
        v[3] = csub(b, id);
    }
};

template <bool INV>
struct Dft<3, INV> {
    static FX_HD void run(float2 (&v)[3])
    {
        constexpr float s3 = INV ? 0.86602540378443865f : -0.86602540378443865f;
        const float2 s = cadd(v[1], v[2]), d = csub(v[1], v[2]);
        const float2 m = make_float2(v[0].x - 0.5f * s.x, v[0].y - 0.5f * s.y);
        const float2 id = make_float2(-s3 * d.y, s3 * d.x);                               // i s3 d
        v[0] = cadd(v[0], s);
        v[1] = cadd(m, id);
        v[2] = csub(m, id);
    }
};

template <bool INV>
struct Dft<5, INV> {
    static FX_HD void run(float2 (&v)[5])
    {
        constexpr float c1 = 0.30901699437494742f, c2 = -0.80901699437494742f;
        constexpr float s1 = INV ? 0.95105651629515357f : -0.95105651629515357f;
        constexpr float s2 = INV ? 0.58778525229247313f : -0.58778525229247313f;
        const float2 a1 = cadd(v[1], v[4]), b1 = csub(v[1], v[4]), a2 = cadd(v[2], v[3]), b2 = csub(v[2], v[3]);
        const float2 m1 = make_float2(v[0].x + c1 * a1.x + c2 * a2.x, v[0].y + c1 * a1.y + c2 * a2.y);
        const float2 m2 = make_float2(v[0].x + c2 * a1.x + c1 * a2.x, v[0].y + c2 * a1.y + c1 * a2.y);
        const float2 n1 = make_float2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
        const float2 n2 = make_float2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
        v[0] = make_float2(v[0].x + a1.x + a2.x, v[0].y + a1.y + a2.y);
        v[1] = make_float2(m1.x - n1.y, m1.y + n1.x);                                       // m1 + i n1
        v[4] = make_float2(m1.x + n1.y, m1.y - n1.x);
        v[2] = make_float2(m2.x - n2.y, m2.y + n2.x);
        v[3] = make_float2(m2.x + n2.y, m2.y - n2.x);
    }
};

}   // namespace fx

// The factorisations the two-step kernels are instantiated for: X(K, N1, N2) with K = N1 N2 the extent of a complex
// axis (x, y), and Z(K2, N1, N2) with K2 = 2 N1 N2 the extent of the real axis (z, transformed as K2/2 complex points).
#define FX_SIZES(X)                                                                                                   \
    X(24, 4, 6) X(32, 8, 4) X(48, 8, 6) X(64, 8, 8) X(72, 8, 9) X(80, 10, 8) X(96, 12, 8) X(108, 12, 9)               \
    X(120, 12, 10) X(128, 16, 8) X(144, 12, 12) X(160, 16, 10) X(192, 16, 12) X(256, 16, 16)
#define FX_ZSIZES(Z)                                                                                                  \
    Z(24, 4, 3) Z(32, 4, 4) Z(48, 4, 6) Z(64, 8, 4) Z(72, 6, 6) Z(80, 8, 5) Z(96, 8, 6) Z(108, 9, 6)                  \
    Z(120, 10, 6) Z(128, 8, 8) Z(144, 9, 8) Z(160, 10, 8) Z(192, 12, 8) Z(256, 16, 8)
