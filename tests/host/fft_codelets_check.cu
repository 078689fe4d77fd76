// Host-side check of the register-resident DFT codelets (paper_2503_21176_b200/csrc/fftx.cuh) and of the index algebra of
// the two-step transforms built on them (fftx.cu: x and y axes; fftz.cu: the real axis as a half-length complex
// transform with an even/odd split), against naive fp64 DFTs written out here.  Compiled by tests/test_fft_host.py with
// nvcc as HOST code (the codelets are __host__ __device__); prints "name max_abs_error" lines.
#include "../../paper_2503_21176_b200/csrc/fftx.cuh"
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstdlib>
#include <vector>
using cd = std::complex<double>;
static const double PI = 3.14159265358979323846;
static float rnd() { return rand() / (float)RAND_MAX - 0.5f; }

template <int N, bool INV> static double dft_err()
{
    float2 v[N];
    cd x[N];
    for (int i = 0; i < N; ++i) { v[i] = make_float2(rnd(), rnd()); x[i] = cd(v[i].x, v[i].y); }
    fx::Dft<N, INV>::run(v);
    double err = 0;
    for (int k = 0; k < N; ++k) {
        cd s = 0;
        for (int n = 0; n < N; ++n) s += x[n] * std::polar(1.0, (INV ? 2.0 : -2.0) * PI * n * k / N);
        err = fmax(err, std::abs(s - cd(v[k].x, v[k].y)));
    }
    return err;
}
template <int N> static void dft_line()
{
    printf("dft%d %.3e\n", N, fmax(dft_err<N, false>(), dft_err<N, true>()));
}

// forward two-step transform of N = N1 N2 points, multiplication by a real G, inverse two-step: as k_xline2 does
template <int N1, int N2> static void two_step()
{
    constexpr int N = N1 * N2;
    std::vector<cd> x(N), X(N), Y(N);
    std::vector<float2> in(N), S(N), W(N);
    std::vector<double> G(N);
    for (int m = 0; m < N; ++m) W[m] = make_float2((float)cos(-2 * PI * m / N), (float)sin(-2 * PI * m / N));
    for (int i = 0; i < N; ++i) { in[i] = make_float2(rnd(), rnd()); x[i] = cd(in[i].x, in[i].y); G[i] = 1.0 / (1.0 + i); }
    for (int k = 0; k < N; ++k) { cd s = 0; for (int n = 0; n < N; ++n) s += x[n] * std::polar(1.0, -2.0 * PI * n * k / N); X[k] = s; }
    for (int n = 0; n < N; ++n) { cd s = 0; for (int k = 0; k < N; ++k) s += G[k] * X[k] * std::polar(1.0, 2.0 * PI * n * k / N); Y[n] = s; }
    for (int n2 = 0; n2 < N2; ++n2) {
        float2 v[N1];
        for (int n1 = 0; n1 < N1; ++n1) v[n1] = in[N2 * n1 + n2];
        fx::Dft<N1, false>::run(v);
        for (int k1 = 0; k1 < N1; ++k1) S[k1 * N2 + n2] = k1 ? fx::cmulf(v[k1], W[n2 * k1]) : v[k1];
    }
    double e1 = 0, e2 = 0;
    for (int k1 = 0; k1 < N1; ++k1) {
        float2 u[N2];
        for (int n2 = 0; n2 < N2; ++n2) u[n2] = S[k1 * N2 + n2];
        fx::Dft<N2, false>::run(u);
        for (int k2 = 0; k2 < N2; ++k2) {
            const int m0 = k1 + N1 * k2;
            e1 = fmax(e1, std::abs(X[m0] - cd(u[k2].x, u[k2].y)));
            u[k2].x *= (float)G[m0]; u[k2].y *= (float)G[m0];
        }
        fx::Dft<N2, true>::run(u);
        for (int n2 = 0; n2 < N2; ++n2) { float2 w = W[k1 * n2]; w.y = -w.y; S[k1 * N2 + n2] = fx::cmulf(u[n2], w); }
    }
    for (int n2 = 0; n2 < N2; ++n2) {
        float2 v[N1];
        for (int k1 = 0; k1 < N1; ++k1) v[k1] = S[k1 * N2 + n2];
        fx::Dft<N1, true>::run(v);
        for (int n1 = 0; n1 < N1; ++n1) e2 = fmax(e2, std::abs(Y[N2 * n1 + n2] - cd(v[n1].x, v[n1].y)));
    }
    printf("twostep%d %.3e\n", N, fmax(e1, e2));
}

// real axis: K2 = 2 M real points as M = N1 N2 complex ones; forward with the even/odd split, inverse with the merge:
// the arithmetic of k_zr2c / k_zc2r for one line
template <int N1, int N2> static void real_axis()
{
    constexpr int M = N1 * N2, K2 = 2 * M;
    std::vector<float> r(K2);
    for (auto& v : r) v = rnd();
    std::vector<cd> X(M + 1), Y(K2);
    for (int k = 0; k <= M; ++k) { cd s = 0; for (int n = 0; n < K2; ++n) s += (double)r[n] * std::polar(1.0, -2.0 * PI * n * k / K2); X[k] = s; }
    std::vector<float2> Wz(K2), S(M), Z(M + 1), Xs(M + 1);
    for (int m = 0; m < K2; ++m) Wz[m] = make_float2((float)cos(-2 * PI * m / K2), (float)sin(-2 * PI * m / K2));
    for (int n2 = 0; n2 < N2; ++n2) {
        float2 v[N1];
        for (int n1 = 0; n1 < N1; ++n1) { const int n = N2 * n1 + n2; v[n1] = make_float2(r[2 * n], r[2 * n + 1]); }
        fx::Dft<N1, false>::run(v);
        for (int k1 = 0; k1 < N1; ++k1) S[k1 * N2 + n2] = k1 ? fx::cmulf(v[k1], Wz[2 * n2 * k1]) : v[k1];
    }
    for (int k1 = 0; k1 < N1; ++k1) {
        float2 u[N2];
        for (int n2 = 0; n2 < N2; ++n2) u[n2] = S[k1 * N2 + n2];
        fx::Dft<N2, false>::run(u);
        for (int k2 = 0; k2 < N2; ++k2) Z[k1 + N1 * k2] = u[k2];
    }
    double e1 = 0, e2 = 0;
    for (int k = 0; k <= M; ++k) {
        const float2 a = Z[k == M ? 0 : k], b = Z[k == 0 ? 0 : M - k];
        const float ex = 0.5f * (a.x + b.x), ey = 0.5f * (a.y - b.y), dx = 0.5f * (a.x - b.x), dy = 0.5f * (a.y + b.y);
        const float2 w = Wz[k];
        const float2 out = make_float2(ex + (dy * w.x + dx * w.y), ey + (dy * w.y - dx * w.x));
        e1 = fmax(e1, std::abs(X[k] - cd(out.x, out.y)));
    }
    // inverse of G X with a real G: expected sum over all K2 frequencies of the Hermitian extension
    for (int k = 0; k <= M; ++k) { Y[k] = X[k] / (1.0 + k); Xs[k] = make_float2((float)Y[k].real(), (float)Y[k].imag()); }
    for (int k = M + 1; k < K2; ++k) Y[k] = std::conj(Y[K2 - k]);
    std::vector<double> want(K2);
    for (int n = 0; n < K2; ++n) { cd s = 0; for (int k = 0; k < K2; ++k) s += Y[k] * std::polar(1.0, 2.0 * PI * n * k / K2); want[n] = s.real(); }
    for (int j = 0; j < N2; ++j) {
        float2 v[N1];
        for (int i = 0; i < N1; ++i) {
            const int k = N2 * i + j;
            const float2 a = Xs[k], b = Xs[M - k], w = Wz[k];
            const float sx = a.x + b.x, sy = a.y - b.y, dx = a.x - b.x, dy = a.y + b.y;
            const float tx = dx * w.x + dy * w.y, ty = dy * w.x - dx * w.y;
            v[i] = make_float2(sx - ty, sy + tx);
        }
        fx::Dft<N1, true>::run(v);
        for (int k1 = 0; k1 < N1; ++k1) { float2 w = Wz[2 * j * k1]; w.y = -w.y; S[k1 * N2 + j] = k1 ? fx::cmulf(v[k1], w) : v[k1]; }
    }
    for (int k1 = 0; k1 < N1; ++k1) {
        float2 u[N2];
        for (int j = 0; j < N2; ++j) u[j] = S[k1 * N2 + j];
        fx::Dft<N2, true>::run(u);
        for (int k2 = 0; k2 < N2; ++k2) {
            const int n = k1 + N1 * k2;
            e2 = fmax(e2, fmax(fabs(want[2 * n] - u[k2].x), fabs(want[2 * n + 1] - u[k2].y)));
        }
    }
    printf("real%d %.3e\n", K2, fmax(e1, e2));
}

int main()
{
    srand(7);
    dft_line<2>(); dft_line<3>(); dft_line<4>(); dft_line<5>(); dft_line<6>(); dft_line<8>(); dft_line<9>(); dft_line<10>();
    dft_line<12>(); dft_line<16>();
#define X(K, N1, N2) two_step<N1, N2>();
    FX_SIZES(X)
#undef X
#define Z(K, N1, N2) real_axis<N1, N2>();
    FX_ZSIZES(Z)
#undef Z
    return 0;
}
