// fftz.cu -- z-axis passes of the PME transforms (a-5 / a-7, Alg. 2 steps 2 and 4): real-to-complex
// forward and complex-to-real inverse of the K2-point lines of the grid, contiguous in memory, as HALF-LENGTH complex
// transforms: z[n] = r[2n] + i r[2n+1], M = K2/2 = N1 N2 points by the register-resident two-step scheme of fftx.cu,
// and the even/odd split
//     Qhat[k] = 1/2 (Z[k] + conj Z[M-k])  -  i/2 e^{-2 pi i k/K2} (Z[k] - conj Z[M-k]),   k = 0..M   (Z[M] = Z[0])
// after it (forward), or its inverse before it (backward, scaled by 2 so that the result is the unnormalised sum
// over all K2 frequencies like cuFFT's C2R).  Lines are dealt TJ to a block; a thread's strided points are N2
// neighbouring threads' contiguous 8-byte elements, so global accesses are runs of 8 N2 bytes on loading and whole
// contiguous tiles on storing.  Unnormalised, layouts as cuFFT's R2C/C2R: grid[line][K2] <-> spec[line][K2/2 + 1].
#include "common.cuh"
#include "fftx.cuh"

namespace {

template <int N1, int N2, int TJ>
struct ZCfg {
    static constexpr int M = N1 * N2, K2 = 2 * M, K2h = M + 1;
    static constexpr int RS = (N2 % 2 == 0) ? N2 + 1 : N2;          // row of one (line, k1): odd stride, no bank conflicts
    static constexpr int ZS = K2h + ((24 - K2h % 16) % 16);          // a line's spectrum, stride = 8 mod 16 elements
    static constexpr int TS = N1 * RS + ((24 - (N1 * RS) % 16) % 16);  // a line's block of S, likewise: the N2-wide runs
                                                                     // of two lines in a half-warp fall on different banks
    static constexpr int NTA = TJ * N2, NTB = TJ * N1;
    static constexpr int NT = (((NTA > NTB ? NTA : NTB) + 31) / 32) * 32;
    static constexpr size_t SMEM = sizeof(float2) * ((size_t)TJ * TS + (size_t)TJ * ZS + K2);
};

template <int N1, int N2, int TJ>
__global__ void __launch_bounds__(ZCfg<N1, N2, TJ>::NT)
k_zr2c(int nlines, const float2* __restrict__ Wg, const float* grid, float2* spec)      // grid: written by the kernel before;
                                                                                    // no __restrict__, or its loads may be hoisted
                                                                                    // above pdl_wait() as read-only (ld.global.nc)
{
    using C = ZCfg<N1, N2, TJ>;
    constexpr int M = C::M, K2 = C::K2, K2h = C::K2h, RS = C::RS, ZS = C::ZS, TS = C::TS, NT = C::NT;
    extern __shared__ __align__(16) float2 z_sh[];                   // S[TJ][N1][RS] | Zs[TJ][ZS] | W[K2]
    float2* S = z_sh;
    float2* Zs = S + TJ * TS;
    float2* W = Zs + TJ * ZS;
    const int tid = threadIdx.x, line0 = blockIdx.x * TJ;
    pdl_trigger();
    for (int i = tid; i < K2; i += NT) W[i] = Wg[i];
    pdl_wait();
    float2 v[N1];
    const int tjA = tid / N2, n2 = tid - tjA * N2;
    const bool actA = tid < C::NTA;
    if (actA) {
        const bool on = line0 + tjA < nlines;
        const float2* src = reinterpret_cast<const float2*>(grid) + (size_t)(line0 + tjA) * M + n2;
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int n1 = decltype(i_)::value;
            v[n1] = on ? src[N2 * n1] : make_float2(0.f, 0.f);
        });
    }
    __syncthreads();
    if (actA) {
        fx::Dft<N1, false>::run(v);
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int k1 = decltype(i_)::value;
            float2 z = v[k1];
            if (k1 > 0) z = fx::cmulf(z, W[2 * n2 * k1]);            // W_M^(n2 k1); 2 n2 k1 < K2
            S[tjA * TS + k1 * RS + n2] = z;
        });
    }
    __syncthreads();
    if (tid < C::NTB) {
        const int tj = tid / N1, k1 = tid - tj * N1;
        float2 u[N2];
        const float2* row = S + tj * TS + k1 * RS;
        fx::sfor<0, N2>([&](auto i_) { constexpr int j = decltype(i_)::value; u[j] = row[j]; });
        fx::Dft<N2, false>::run(u);
        fx::sfor<0, N2>([&](auto i_) { constexpr int k2 = decltype(i_)::value; Zs[tj * ZS + k1 + N1 * k2] = u[k2]; });
    }
    __syncthreads();
    // even/odd split and the store of the tile's TJ * K2h contiguous outputs
    const int nout = min(TJ, nlines - line0) * K2h;
    float2* dst = spec + (size_t)line0 * K2h;
    for (int e = tid; e < nout; e += NT) {
        const int tj = e / K2h, k = e - tj * K2h;
        const float2 a = Zs[tj * ZS + (k == M ? 0 : k)], b = Zs[tj * ZS + (k == 0 ? 0 : M - k)];
        const float ex = 0.5f * (a.x + b.x), ey = 0.5f * (a.y - b.y);           // 1/2 (a + conj b)
        const float dx = 0.5f * (a.x - b.x), dy = 0.5f * (a.y + b.y);           // 1/2 (a - conj b)
        const float2 w = W[k];
        // -i d w = (dy, -dx) * w
        dst[e] = make_float2(ex + (dy * w.x + dx * w.y), ey + (dy * w.y - dx * w.x));
    }
}

template <int N1, int N2, int TJ>
__global__ void __launch_bounds__(ZCfg<N1, N2, TJ>::NT)
k_zc2r(int nlines, const float2* __restrict__ Wg, const float2* spec, float* grid)      // spec: likewise
{
    using C = ZCfg<N1, N2, TJ>;
    constexpr int M = C::M, K2 = C::K2, K2h = C::K2h, RS = C::RS, ZS = C::ZS, TS = C::TS, NT = C::NT;
    extern __shared__ __align__(16) float2 z_sh[];
    float2* S = z_sh;
    float2* W = S + TJ * TS + TJ * ZS;
    const int tid = threadIdx.x, line0 = blockIdx.x * TJ;
    pdl_trigger();
    for (int i = tid; i < K2; i += NT) W[i] = Wg[i];
    pdl_wait();
    // the even/odd merge needs Qhat[k] and Qhat[M-k]: both straight from global memory (each element is read by two
    // threads of the block; the second read hits L1)
    const int tjA = tid / N2, j = tid - tjA * N2;
    const bool actA = tid < C::NTA && line0 + tjA < nlines;
    float2 xa[N1], xb[N1];
    if (actA) {
        const float2* X = spec + (size_t)(line0 + tjA) * K2h;
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int i = decltype(i_)::value;
            xa[i] = X[N2 * i + j];
            xb[i] = X[M - N2 * i - j];
        });
    }
    __syncthreads();                                                  // W
    if (tid < C::NTA) {
        float2 v[N1];
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int i = decltype(i_)::value;
            const int k = N2 * i + j;
            const float2 a = actA ? xa[i] : make_float2(0.f, 0.f), b = actA ? xb[i] : make_float2(0.f, 0.f);
            const float sx = a.x + b.x, sy = a.y - b.y;                            // a + conj b
            const float dx = a.x - b.x, dy = a.y + b.y;                            // a - conj b
            const float2 w = W[k];                                                 // conj w below
            const float tx = dx * w.x + dy * w.y, ty = dy * w.x - dx * w.y;        // d conj(w)
            v[i] = make_float2(sx - ty, sy + tx);                                  // s + i t
        });
        fx::Dft<N1, true>::run(v);
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int k1 = decltype(i_)::value;
            float2 z = v[k1];
            if (k1 > 0) {
                float2 c = W[2 * j * k1];
                c.y = -c.y;
                z = fx::cmulf(z, c);
            }
            S[tjA * TS + k1 * RS + j] = z;
        });
    }
    __syncthreads();
    if (tid < C::NTB) {
        const int tj = tid / N1, k1 = tid - tj * N1;
        float2 u[N2];
        const float2* row = S + tj * TS + k1 * RS;
        fx::sfor<0, N2>([&](auto i_) { constexpr int jj = decltype(i_)::value; u[jj] = row[jj]; });
        fx::Dft<N2, true>::run(u);
        if (line0 + tj < nlines) {
            float2* dst = reinterpret_cast<float2*>(grid) + (size_t)(line0 + tj) * M + k1;
            fx::sfor<0, N2>([&](auto i_) { constexpr int k2 = decltype(i_)::value; dst[N1 * k2] = u[k2]; });
        }
    }
}

template <int N1, int N2, int TJ>
int launch_z(sqeq_ctx* ctx, int nlines, const float2* W, float* grid, float2* spec, bool inverse, cudaStream_t st)
{
    using C = ZCfg<N1, N2, TJ>;
    const int nb = ceil_div(nlines, TJ);
    if (inverse) {
        auto kern = k_zc2r<N1, N2, TJ>;
        CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        CUDA_TRY(ctx, launch_pdl(ctx, kern, dim3(nb), dim3(C::NT), C::SMEM, st, nlines, W, spec, grid));
    } else {
        auto kern = k_zr2c<N1, N2, TJ>;
        CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        CUDA_TRY(ctx, launch_pdl(ctx, kern, dim3(nb), dim3(C::NT), C::SMEM, st, nlines, W, (const float*)grid, spec));
    }
    return SQEQ_OK;
}

}   // namespace

bool zline_supported(int K2)
{
    switch (K2) {
#define FX_CASE(KK, N1, N2) case KK:
        FX_ZSIZES(FX_CASE) return true;
#undef FX_CASE
    default: return false;
    }
}

// forward: grid[nlines][K2] (real) -> spec[nlines][K2/2+1]; inverse: the other way.  W = the K2-th roots of unity.
int zline_run(sqeq_ctx* ctx, int nlines, int K2, const float2* W, float* grid, float2* spec, bool inverse, cudaStream_t st)
{
    switch (K2) {
#define FX_CASE(KK, N1, N2) case KK: return launch_z<N1, N2, 16>(ctx, nlines, W, grid, spec, inverse, st);
        FX_ZSIZES(FX_CASE)
#undef FX_CASE
    default: return sqeq_fail(ctx, SQEQ_EINVAL, "zline_run: unsupported z extent %d", K2);
    }
}
