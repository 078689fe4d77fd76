// fftx.cu -- the fused x-axis pass of the PME reciprocal part, register-resident two-step version.
//
// north_star: "the influence-function convolution fused into the FFT pre- and post-passes" (Alg. 2 steps 2-4,
// PAPER.md:147-149).  The 3-D transforms are split as  [z real-to-complex (fftz.cu), y forward (k_yline below); or a
// batched 2-D cuFFT R2C over (y,z)] -> k_xline2 -> [y inverse, z complex-to-real; or cuFFT 2-D C2R].  k_xline2
// does, for a tile of TJ neighbouring (m1, m2) lines, the forward transform along x, the
// multiplication by G(m) with the energy sum, and the inverse transform along x, reading and writing the spectrum
// once.  K0 = N1 * N2 with N1, N2 <= 16, and each transform is TWO register-resident DFTs (fftx.cuh) around ONE
// exchange through shared memory:
//
//   forward   x = N2 n1 + n2,  m0 = k1 + N1 k2:
//     thread (n2, line): loads its N1 points straight from global memory, DFT-N1 over n1, times W_N^(n2 k1) -> shared
//     thread (k1, line): DFT-N2 over n2 -> Qhat(m0 = k1 + N1 k2), k2 in registers
//   influence  Qhat *= G, E += w G |Qhat|^2                          (same registers)
//   inverse   the same decomposition run backwards:
//     thread (k1, line): inverse DFT-N2 over k2, times conj W_N^(k1 n2) -> the SAME shared slots it read
//     thread (n2, line): inverse DFT-N1 over k1 -> Phi-hat(x = N2 n1 + n2), stored straight to global memory
//
// Two block-wide barriers per tile; about a third of the instructions of the radix-2/3/4/5 Stockham version in
// pme.cu (k_xline_influence, kept for grid sizes that do not factor this way).
#include "common.cuh"
#include "fftx.cuh"

namespace {

template <int N1, int N2, int TJ>
struct XlCfg {
    static constexpr int N = N1 * N2;
    static constexpr int NT = (((N1 > N2 ? N1 : N2) * TJ + 31) / 32) * 32;      // whole warps; the surplus threads idle
    // 64-bit shared accesses go out per half-warp (16 lanes).  Step-B threads (k1, line) are TJ lines x 16/TJ values
    // of k1 per half-warp: the k1 stride must put those on different banks.
    static constexpr int PAD = (TJ >= 16) ? 0 : (((N2 * TJ) % 16 == 0) ? TJ : 0);
    static constexpr int SK1 = N2 * TJ + PAD;               // float2 elements per k1 row
    static constexpr size_t SMEM = sizeof(float2) * ((size_t)N1 * SK1 + N);
};

template <int N1, int N2, int TJ>
__global__ void __launch_bounds__(XlCfg<N1, N2, TJ>::NT)
k_xline2(int K1, int K2h, int K2, const float* __restrict__ tab, float inv_piV, const float2* __restrict__ Wg,
         float2* __restrict__ spec, double* __restrict__ e_out)
{
    using C = XlCfg<N1, N2, TJ>;
    constexpr int N = C::N, NT = C::NT, SK1 = C::SK1;
    extern __shared__ __align__(16) float2 xl_sh[];         // S[N1][SK1] | W[N]
    float2* S = xl_sh;
    float2* W = S + N1 * SK1;
    const int nline = K1 * K2h;
    const int tid = threadIdx.x, tj = tid % TJ, hi = tid / TJ;     // hi = n2 (steps A, A') or k1 (step B)
    const int jl = blockIdx.x * TJ + tj;
    const bool line_on = jl < nline;
    pdl_trigger();
    for (int i = tid; i < N; i += NT) W[i] = Wg[i];
    pdl_wait();

    // ---- step A: N1-point transforms over n1, straight from global memory
    float2 v[N1];
    const bool actA = hi < N2;
    if (actA) {
        float2* g = spec + (size_t)hi * nline + jl;
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int n1 = decltype(i_)::value;
            v[n1] = line_on ? g[(size_t)(N2 * n1) * nline] : make_float2(0.f, 0.f);
        });
    }
    __syncthreads();                                        // W is there
    if (actA) {
        fx::Dft<N1, false>::run(v);
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int k1 = decltype(i_)::value;
            float2 z = v[k1];
            if (k1 > 0) z = fx::cmulf(z, W[hi * k1]);       // n2 k1 < N
            S[k1 * SK1 + hi * TJ + tj] = z;
        });
    }
    __syncthreads();

    // ---- step B: N2-point transforms over n2, influence function, inverse N2-point transforms over k2
    float er = 0.f;
    if (hi < N1) {
        float2 u[N2];
        float2* row = S + hi * SK1 + tj;
        fx::sfor<0, N2>([&](auto i_) { constexpr int n2 = decltype(i_)::value; u[n2] = row[n2 * TJ]; });
        fx::Dft<N2, false>::run(u);
        // G(m) as in k_influence / k_xline_influence (pme.cu); the line's (m1, m2) factors once per thread
        const float* Bg0 = tab;       const float* s0 = Bg0 + N;
        const float* Bg1 = s0 + N;    const float* s1 = Bg1 + K1;
        const float* Bg2 = s1 + K1;   const float* s2 = Bg2 + K2;
        const int m1 = line_on ? jl / K2h : 0, m2 = line_on ? jl - m1 * K2h : 0;
        const float bg12 = Bg1[m1] * Bg2[m2] * inv_piV, s12 = s1[m1] + s2[m2];
        const float w = !line_on ? 0.f : ((m2 == 0 || 2 * m2 == K2) ? 0.5f : 1.0f);
        fx::sfor<0, N2>([&](auto i_) {
            constexpr int k2 = decltype(i_)::value;
            const int m0 = hi + N1 * k2;
            float G = 0.f;
            if (line_on && (m0 | jl)) G = __fdividef(__ldg(Bg0 + m0) * bg12, __ldg(s0 + m0) + s12);
            float2 z = u[k2];
            er = fmaf(w * G, fmaf(z.x, z.x, z.y * z.y), er);
            u[k2] = make_float2(z.x * G, z.y * G);
        });
        fx::Dft<N2, true>::run(u);
        fx::sfor<0, N2>([&](auto i_) {
            constexpr int n2 = decltype(i_)::value;
            float2 z = u[n2];
            if (n2 > 0) {
                float2 c = W[hi * n2];                      // k1 n2 < N
                c.y = -c.y;
                z = fx::cmulf(z, c);
            }
            row[n2 * TJ] = z;                               // the slots this thread read: no barrier needed before
        });
    }
    __syncthreads();

    // ---- step A': inverse N1-point transforms over k1, straight to global memory
    if (actA) {
        fx::sfor<0, N1>([&](auto i_) { constexpr int k1 = decltype(i_)::value; v[k1] = S[k1 * SK1 + hi * TJ + tj]; });
        fx::Dft<N1, true>::run(v);
        if (line_on) {
            float2* g = spec + (size_t)hi * nline + jl;
            fx::sfor<0, N1>([&](auto i_) { constexpr int n1 = decltype(i_)::value; g[(size_t)(N2 * n1) * nline] = v[n1]; });
        }
    }
    if (e_out) {
        double e = (double)er;
        __shared__ double red[NT / 32 + 1];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        if ((tid & 31) == 0) red[tid >> 5] = e;
        __syncthreads();
        if (tid == 0) {
            double t = 0.0;
            for (int k = 0; k < (NT + 31) / 32; ++k) t += red[k];
            atomicAdd(e_out, t);
        }
    }
}

template <int N1, int N2, int TJ>
int launch(sqeq_ctx* ctx, int K1, int K2h, int K2, const float* tab, float inv_piV, const float2* W, float2* spec,
           double* e_out, cudaStream_t st)
{
    using C = XlCfg<N1, N2, TJ>;
    static_assert(C::NT % 32 == 0 && C::NT <= 1024, "whole warps");
    auto kern = k_xline2<N1, N2, TJ>;
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    CUDA_TRY(ctx, launch_pdl(ctx, kern, dim3(ceil_div((int64_t)K1 * K2h, TJ)), dim3(C::NT), C::SMEM, st, K1, K2h, K2, tab, inv_piV, W, spec,
                             e_out));
    return SQEQ_OK;
}

// ---- y-axis pass: plain forward or inverse transform of the lines (x, ., zc), stride K2h, in place.  Same two-step
// scheme; the second step stores straight to global memory, so there is one data barrier.
template <int N1, int N2, int TJ, bool INV>
__global__ void __launch_bounds__(XlCfg<N1, N2, TJ>::NT)
k_yline(int K2h, const float2* __restrict__ Wg, float2* __restrict__ spec)
{
    using C = XlCfg<N1, N2, TJ>;
    constexpr int N = C::N, NT = C::NT, SK1 = C::SK1;
    extern __shared__ __align__(16) float2 xl_sh[];         // S[N1][SK1] | W[N]
    float2* S = xl_sh;
    float2* W = S + N1 * SK1;
    const int tid = threadIdx.x, tj = tid % TJ, hi = tid / TJ;
    const int zc = blockIdx.x * TJ + tj;
    const bool line_on = zc < K2h;
    float2* g = spec + (size_t)blockIdx.y * N * K2h + zc;   // (x, y = 0, zc)
    pdl_trigger();
    for (int i = tid; i < N; i += NT) W[i] = Wg[i];
    pdl_wait();
    float2 v[N1];
    const bool actA = hi < N2;
    if (actA) {
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int n1 = decltype(i_)::value;
            v[n1] = line_on ? g[(size_t)(N2 * n1 + hi) * K2h] : make_float2(0.f, 0.f);
        });
    }
    __syncthreads();
    if (actA) {
        fx::Dft<N1, INV>::run(v);
        fx::sfor<0, N1>([&](auto i_) {
            constexpr int k1 = decltype(i_)::value;
            float2 z = v[k1];
            if (k1 > 0) {
                float2 c = W[hi * k1];
                if (INV) c.y = -c.y;
                z = fx::cmulf(z, c);
            }
            S[k1 * SK1 + hi * TJ + tj] = z;
        });
    }
    __syncthreads();
    if (hi < N1) {
        float2 u[N2];
        const float2* row = S + hi * SK1 + tj;
        fx::sfor<0, N2>([&](auto i_) { constexpr int n2 = decltype(i_)::value; u[n2] = row[n2 * TJ]; });
        fx::Dft<N2, INV>::run(u);
        if (line_on)
            fx::sfor<0, N2>([&](auto i_) { constexpr int k2 = decltype(i_)::value; g[(size_t)(hi + N1 * k2) * K2h] = u[k2]; });
    }
}

template <int N1, int N2, int TJ>
int launch_y(sqeq_ctx* ctx, int K0, int K2h, const float2* W, float2* spec, bool inverse, cudaStream_t st)
{
    using C = XlCfg<N1, N2, TJ>;
    const dim3 gr((unsigned)ceil_div(K2h, TJ), (unsigned)K0);
    if (inverse) {
        auto kern = k_yline<N1, N2, TJ, true>;
        CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        CUDA_TRY(ctx, launch_pdl(ctx, kern, gr, dim3(C::NT), C::SMEM, st, K2h, W, spec));
    } else {
        auto kern = k_yline<N1, N2, TJ, false>;
        CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        CUDA_TRY(ctx, launch_pdl(ctx, kern, gr, dim3(C::NT), C::SMEM, st, K2h, W, spec));
    }
    return SQEQ_OK;
}

}   // namespace

// The x (and y) extents this file is built for.
bool xline2_supported(int K)
{
    switch (K) {
#define FX_CASE(KK, N1, N2) case KK:
        FX_SIZES(FX_CASE) return true;
#undef FX_CASE
    default: return false;
    }
}

int xline2_run(sqeq_ctx* ctx, int K0, int K1, int K2h, int K2, const float* tab, float inv_piV, const float2* W,
               float2* spec, double* e_out, cudaStream_t st)
{
    switch (K0) {
#define FX_CASE(KK, N1, N2) case KK: return launch<N1, N2, 16>(ctx, K1, K2h, K2, tab, inv_piV, W, spec, e_out, st);
        FX_SIZES(FX_CASE)
#undef FX_CASE
    default: return sqeq_fail(ctx, SQEQ_EINVAL, "xline2_run: unsupported x extent %d", K0);
    }
}

// forward or inverse transform along y of spec[K0][K1][K2h], in place; W = the K1-th roots of unity e^{-2 pi i m/K1}
int yline_run(sqeq_ctx* ctx, int K0, int K1, int K2h, const float2* W, float2* spec, bool inverse, cudaStream_t st)
{
    switch (K1) {
#define FX_CASE(KK, N1, N2) case KK: return launch_y<N1, N2, 16>(ctx, K0, K2h, W, spec, inverse, st);
        FX_SIZES(FX_CASE)
#undef FX_CASE
    default: return sqeq_fail(ctx, SQEQ_EINVAL, "yline_run: unsupported y extent %d", K1);
    }
}
