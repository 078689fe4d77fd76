// pme.cu -- smooth Particle Mesh Ewald, Alg. 2, steps a-4 ... a-8:
//   spread (order-p cardinal B-splines) -> cuFFT R2C -> influence multiply (+ E_rec) -> cuFFT C2R
//   -> gather of phi_rec and F_rec.  Conventions are DESIGN.md R-PME: weight M_p(w+j) on grid index
//   f-j, unnormalised transforms (no 1/K^3), G(m) = B(m) exp(-pi^2 mt^2/alpha^2)/(pi V mt^2), G(0)=0.
// cuFFT does the two 3-D transforms (north_star allows it; timed as separate stages).
#include <math.h>

#include <vector>

#include "common.cuh"

// -------------------------------------------------------------------------------------- weights
// theta[j] = M_P(w + j), dtheta[j] = M_P'(w + j), j = 0..P-1, by the cardinal B-spline recursion
//   M_n(u) = [u M_{n-1}(u) + (n-u) M_{n-1}(u-1)]/(n-1),  M_n'(u) = M_{n-1}(u) - M_{n-1}(u-1).
template <int P>
__device__ __forceinline__ void bspline_weights(float w, float* theta, float* dtheta)
{
    float a[P];
#pragma unroll
    for (int j = 0; j < P; ++j) a[j] = 0.f;
    a[0] = w;          // M_2(w)
    a[1] = 1.f - w;    // M_2(w+1)
#pragma unroll
    for (int n = 3; n <= P; ++n) {
        if (n == P) {
#pragma unroll
            for (int j = 0; j < P; ++j) dtheta[j] = a[j] - (j > 0 ? a[j - 1] : 0.f);
        }
        const float inv = 1.f / (float)(n - 1);
#pragma unroll
        for (int j = n - 1; j >= 0; --j) {
            const float lo = j > 0 ? a[j - 1] : 0.f;
            a[j] = ((w + (float)j) * a[j] + ((float)n - w - (float)j) * lo) * inv;
        }
    }
#pragma unroll
    for (int j = 0; j < P; ++j) theta[j] = a[j];
}

// -------------------------------------------------------------------------------------- spread
// a-4, Alg. 2 step 1.  One warp per atom; lanes 0..2 evaluate the three axes'
// weights into shared memory, then the 32 lanes sweep the P^3 points z-fastest (contiguous rows of P
// floats) and reduce into the grid with red.global.add.f32.
template <int P>
__global__ void __launch_bounds__(256)
k_spread(int64_t n, const float4* __restrict__ frac, const int4* __restrict__ base, int K0, int K1, int K2,
         float* __restrict__ grid)
{
    __shared__ float wt[8][3][P];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t s = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (s >= n) return;
    const float4 fw = frac[s];
    const int4 f = base[s];
    if (lane < 3) {
        float th[P], dth[P];
        bspline_weights<P>(lane == 0 ? fw.x : (lane == 1 ? fw.y : fw.z), th, dth);
#pragma unroll
        for (int j = 0; j < P; ++j) wt[wid][lane][j] = th[j];
    }
    __syncwarp();
    if (fw.w == 0.f) return;
    for (int pidx = lane; pidx < P * P * P; pidx += 32) {
        const int c = pidx % P, b = (pidx / P) % P, a = pidx / (P * P);
        int gx = f.x - a; gx += gx < 0 ? K0 : 0;
        int gy = f.y - b; gy += gy < 0 ? K1 : 0;
        int gz = f.z - c; gz += gz < 0 ? K2 : 0;
        const float v = fw.w * wt[wid][0][a] * wt[wid][1][b] * wt[wid][2][c];
        atomicAdd(grid + ((size_t)gx * K1 + gy) * K2 + gz, v);
    }
}

// -------------------------------------------------------------------------------------- influence
// a-6, Alg. 2 step 3: Qhat(m) *= G(m); E_rec = 1/2 sum_m G |Qhat|^2 with Hermitian
// weights on the half spectrum.  G is formed in fp64 from three per-axis tables.
__global__ void __launch_bounds__(256)
k_influence(int K0, int K1, int K2h, int K2, const double* __restrict__ tab, double inv_piV,
            float2* __restrict__ spec, double* __restrict__ e_out)
{
    const int64_t total = (int64_t)K0 * K1 * K2h;
    const double* B0 = tab;               const double* g0 = B0 + K0;  const double* s0 = g0 + K0;
    const double* B1 = s0 + K0;           const double* g1 = B1 + K1;  const double* s1 = g1 + K1;
    const double* B2 = s1 + K1;           const double* g2 = B2 + K2;  const double* s2 = g2 + K2;
    double e = 0.0;
    for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int m2 = (int)(idx % K2h);
        const int m1 = (int)((idx / K2h) % K1);
        const int m0 = (int)(idx / ((int64_t)K2h * K1));
        double G = 0.0;
        if (m0 | m1 | m2) {
            const double mt2 = s0[m0] + s1[m1] + s2[m2];
            G = B0[m0] * B1[m1] * B2[m2] * g0[m0] * g1[m1] * g2[m2] * inv_piV / mt2;
        }
        float2 z = spec[idx];
        const double w = (m2 == 0 || 2 * m2 == K2) ? 0.5 : 1.0;     // 1/2 * (1 or 2)
        e += w * G * ((double)z.x * z.x + (double)z.y * z.y);
        const float Gf = (float)G;
        z.x *= Gf;
        z.y *= Gf;
        spec[idx] = z;
    }
    if (e_out) {
        __shared__ double red[8];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e;
        __syncthreads();
        if (threadIdx.x < 8) {
            e = red[threadIdx.x];
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) e += __shfl_xor_sync(0xffu, e, o);
            if (threadIdx.x == 0) atomicAdd(e_out, e);
        }
    }
}

// -------------------------------------------------------------------------------------- gather
// a-8, Alg. 2 step 5: phi_i = sum W Phi;  F_i,x = -q_i (K_x/L_x) sum dW_x Phi.
template <int P, bool FORCE>
__global__ void __launch_bounds__(256)
k_gather(int64_t n, const float4* __restrict__ frac, const int4* __restrict__ base, int K0, int K1, int K2,
         const float* __restrict__ grid, float sx, float sy, float sz, float4* __restrict__ out)
{
    __shared__ float wt[8][6][P];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t s = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (s >= n) return;
    const float4 fw = frac[s];
    const int4 f = base[s];
    if (lane < 3) {
        float th[P], dth[P];
        bspline_weights<P>(lane == 0 ? fw.x : (lane == 1 ? fw.y : fw.z), th, dth);
#pragma unroll
        for (int j = 0; j < P; ++j) { wt[wid][lane][j] = th[j]; wt[wid][3 + lane][j] = dth[j]; }
    }
    __syncwarp();
    float ph = 0.f, gx_ = 0.f, gy_ = 0.f, gz_ = 0.f;
    for (int pidx = lane; pidx < P * P * P; pidx += 32) {
        const int c = pidx % P, b = (pidx / P) % P, a = pidx / (P * P);
        int gx = f.x - a; gx += gx < 0 ? K0 : 0;
        int gy = f.y - b; gy += gy < 0 ? K1 : 0;
        int gz = f.z - c; gz += gz < 0 ? K2 : 0;
        const float v = __ldg(grid + ((size_t)gx * K1 + gy) * K2 + gz);
        const float tx = wt[wid][0][a], ty = wt[wid][1][b], tz = wt[wid][2][c];
        ph = fmaf(tx * ty * tz, v, ph);
        if (FORCE) {
            gx_ = fmaf(wt[wid][3][a] * ty * tz, v, gx_);
            gy_ = fmaf(tx * wt[wid][4][b] * tz, v, gy_);
            gz_ = fmaf(tx * ty * wt[wid][5][c], v, gz_);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ph += __shfl_xor_sync(0xffffffffu, ph, o);
        if (FORCE) {
            gx_ += __shfl_xor_sync(0xffffffffu, gx_, o);
            gy_ += __shfl_xor_sync(0xffffffffu, gy_, o);
            gz_ += __shfl_xor_sync(0xffffffffu, gz_, o);
        }
    }
    if (lane == 0) out[s] = make_float4(-sx * gx_, -sy * gy_, -sz * gz_, ph);   // per unit charge; a-9 applies q_i
}

// -------------------------------------------------------------------------------------- host side
static double host_bspline(int n, double u)
{
    if (n == 2) return (u < 0.0 || u > 2.0) ? 0.0 : 1.0 - fabs(u - 1.0);
    return (u * host_bspline(n - 1, u) + (n - u) * host_bspline(n - 1, u - 1.0)) / (n - 1);
}

int pme_setup(sqeq_ctx* ctx, const double box[3], double alpha, const int grid[3], int order)
{
    const bool same_grid = ctx->plans_ok && grid[0] == ctx->K[0] && grid[1] == ctx->K[1] && grid[2] == ctx->K[2];
    const bool same_tabs = same_grid && order == ctx->order && alpha == ctx->tab_alpha &&
                           box[0] == ctx->tab_box[0] && box[1] == ctx->tab_box[1] && box[2] == ctx->tab_box[2];
    if (same_tabs) return SQEQ_OK;
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream2));
    if (!same_grid) {
        if (ctx->plans_ok) {
            cufftDestroy(ctx->plan_r2c);
            cufftDestroy(ctx->plan_c2r);
            ctx->plans_ok = false;
        }
        cufftResult r = cufftPlan3d(&ctx->plan_r2c, grid[0], grid[1], grid[2], CUFFT_R2C);
        if (r != CUFFT_SUCCESS) return sqeq_fail(ctx, SQEQ_ECUFFT, "cufftPlan3d(R2C %dx%dx%d) failed: %d", grid[0], grid[1], grid[2], (int)r);
        r = cufftPlan3d(&ctx->plan_c2r, grid[0], grid[1], grid[2], CUFFT_C2R);
        if (r != CUFFT_SUCCESS) {
            cufftDestroy(ctx->plan_r2c);
            return sqeq_fail(ctx, SQEQ_ECUFFT, "cufftPlan3d(C2R) failed: %d", (int)r);
        }
        ctx->plans_ok = true;
        for (int d = 0; d < 3; ++d) ctx->K[d] = grid[d];
        const size_t G3 = (size_t)grid[0] * grid[1] * grid[2];
        const size_t S3 = (size_t)grid[0] * grid[1] * (grid[2] / 2 + 1);
        SQEQ_TRY(sqeq_reserve(ctx, ctx->grid, sizeof(float) * G3));
        SQEQ_TRY(sqeq_reserve(ctx, ctx->spec, sizeof(float2) * S3));
    }
    // per-axis tables: |b(m)|^2, exp(-pi^2 mt^2/alpha^2), mt^2   (DESIGN.md R-PME)
    const int Ksum = grid[0] + grid[1] + grid[2];
    std::vector<double> tab(3 * (size_t)Ksum);
    size_t off = 0;
    for (int d = 0; d < 3; ++d) {
        const int K = grid[d];
        double* B = tab.data() + off; double* g = B + K; double* s = g + K;
        for (int m = 0; m < K; ++m) {
            double re = 0, im = 0;
            for (int k = 0; k <= order - 2; ++k) {
                double a = 2.0 * M_PI * (double)m * (double)k / (double)K;
                double M = host_bspline(order, (double)(k + 1));
                re += M * cos(a);
                im += M * sin(a);
            }
            B[m] = 1.0 / (re * re + im * im);
            double mp = (m <= K / 2 ? m : m - K) / box[d];
            s[m] = mp * mp;
            g[m] = exp(-M_PI * M_PI * mp * mp / (alpha * alpha));
        }
        off += 3 * (size_t)K;
    }
    SQEQ_TRY(sqeq_reserve(ctx, ctx->tabs, sizeof(double) * tab.size()));
    CUDA_TRY(ctx, cudaMemcpy(ctx->tabs.p, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice));
    ctx->order = order;
    ctx->tab_alpha = alpha;
    for (int d = 0; d < 3; ++d) ctx->tab_box[d] = box[d];
    return SQEQ_OK;
}

template <int P>
static int pme_run_t(sqeq_ctx* ctx, int64_t n, const double box[3], bool want_force, bool want_energy,
                     cudaStream_t st)
{
    const int K0 = ctx->K[0], K1 = ctx->K[1], K2 = ctx->K[2], K2h = K2 / 2 + 1;
    const size_t G3 = (size_t)K0 * K1 * K2;
    float* grid = (float*)ctx->grid.p;
    float2* spec = (float2*)ctx->spec.p;
    const float4* frac = (const float4*)ctx->frac.p;
    const int4* base = (const int4*)ctx->base.p;
    SQEQ_TRY(sqeq_reserve(ctx, ctx->rec_out, sizeof(float4) * n));
    const int nbw = ceil_div(n * 32, 256);
    {
        StageTimer tm(ctx, SQEQ_T_SPREAD, st);
        CUDA_TRY(ctx, cudaMemsetAsync(grid, 0, sizeof(float) * G3, st));
        k_spread<P><<<nbw, 256, 0, st>>>(n, frac, base, K0, K1, K2, grid);
        KERNEL_CHECK(ctx);
    }
    if (ctx->gridQ.p) CUDA_TRY(ctx, cudaMemcpyAsync(ctx->gridQ.p, grid, sizeof(float) * G3, cudaMemcpyDeviceToDevice, st));
    {
        StageTimer tm(ctx, SQEQ_T_FFT_FWD, st);
        cufftSetStream(ctx->plan_r2c, st);
        cufftResult r = cufftExecR2C(ctx->plan_r2c, grid, (cufftComplex*)spec);
        if (r != CUFFT_SUCCESS) return sqeq_fail(ctx, SQEQ_ECUFFT, "cufftExecR2C failed: %d", (int)r);
    }
    {
        StageTimer tm(ctx, SQEQ_T_INFLUENCE, st);
        double* e_out = (double*)ctx->scal.p + 1;
        CUDA_TRY(ctx, cudaMemsetAsync(e_out, 0, sizeof(double), st));
        const double inv_piV = 1.0 / (M_PI * box[0] * box[1] * box[2]);
        const int64_t total = (int64_t)K0 * K1 * K2h;
        int nb = ceil_div(total, 256);
        if (nb > ctx->sm_count * 8) nb = ctx->sm_count * 8;
        k_influence<<<nb, 256, 0, st>>>(K0, K1, K2h, K2, (const double*)ctx->tabs.p, inv_piV, spec, e_out);
        KERNEL_CHECK(ctx);
    }
    {
        StageTimer tm(ctx, SQEQ_T_FFT_INV, st);
        cufftSetStream(ctx->plan_c2r, st);
        cufftResult r = cufftExecC2R(ctx->plan_c2r, (cufftComplex*)spec, grid);
        if (r != CUFFT_SUCCESS) return sqeq_fail(ctx, SQEQ_ECUFFT, "cufftExecC2R failed: %d", (int)r);
    }
    {
        StageTimer tm(ctx, SQEQ_T_GATHER, st);
        const float sx = (float)(K0 / box[0]), sy = (float)(K1 / box[1]), sz = (float)(K2 / box[2]);
        if (want_force)
            k_gather<P, true><<<nbw, 256, 0, st>>>(n, frac, base, K0, K1, K2, grid, sx, sy, sz, (float4*)ctx->rec_out.p);
        else
            k_gather<P, false><<<nbw, 256, 0, st>>>(n, frac, base, K0, K1, K2, grid, sx, sy, sz, (float4*)ctx->rec_out.p);
        KERNEL_CHECK(ctx);
    }
    (void)want_energy;
    return SQEQ_OK;
}

int pme_run(sqeq_ctx* ctx, int64_t n, const double box[3], bool want_force, bool want_energy,
            cudaStream_t st)
{
    switch (ctx->order) {
        case 4: return pme_run_t<4>(ctx, n, box, want_force, want_energy, st);
        case 6: return pme_run_t<6>(ctx, n, box, want_force, want_energy, st);
        case 8: return pme_run_t<8>(ctx, n, box, want_force, want_energy, st);
    }
    return sqeq_fail(ctx, SQEQ_EINVAL, "pme_run: unsupported order %d", ctx->order);
}

// -------------------------------------------------------------------------------------- diagnostics
__global__ void k_unpermute_parts(int64_t n, const float4* __restrict__ src, const float4* __restrict__ xq,
                                  const int* __restrict__ perm, float* __restrict__ phi, float* __restrict__ F)
{
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= n) return;
    const float4 v = src[s];
    const float qi = xq[s].w;
    const int64_t o = perm[s];
    if (phi) phi[o] = v.w;
    if (F) { F[3 * o] = qi * v.x; F[3 * o + 1] = qi * v.y; F[3 * o + 2] = qi * v.z; }
}

extern "C" int sqeq_coulomb_parts(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, float* phi_real,
                                  float* F_real, float* phi_rec, float* F_rec, double* E_rec)
{
    if (!ctx || !nl || nl->ctx != ctx || n != nl->n || ctx->last_n != n)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_parts: no matching previous sqeq_coulomb call");
    if ((F_real || F_rec) && !ctx->last_had_force)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_parts: the last evaluation was potential-only");
    cudaStream_t st = ctx->stream;
    k_unpermute_parts<<<ceil_div(n, 256), 256, 0, st>>>(n, (const float4*)ctx->real_out.p, (const float4*)ctx->xq.p, nl->perm, phi_real, F_real);
    KERNEL_CHECK(ctx);
    k_unpermute_parts<<<ceil_div(n, 256), 256, 0, st>>>(n, (const float4*)ctx->rec_out.p, (const float4*)ctx->xq.p, nl->perm, phi_rec, F_rec);
    KERNEL_CHECK(ctx);
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal + 8, (double*)ctx->scal.p + 1, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if (E_rec) *E_rec = ctx->h_scal[8];
    return SQEQ_OK;
}

extern "C" int sqeq_pme_grid(sqeq_ctx* ctx, int which, float* out)
{
    if (!ctx || !out || !ctx->plans_ok) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_pme_grid: no PME state");
    const size_t G3 = (size_t)ctx->K[0] * ctx->K[1] * ctx->K[2];
    if (which == 0) {
        if (!ctx->gridQ.p) {
            // first request: start keeping a copy of Q from the next evaluation on
            SQEQ_TRY(sqeq_reserve(ctx, ctx->gridQ, sizeof(float) * G3));
            return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_pme_grid: Q capture enabled; run sqeq_coulomb again, then re-read");
        }
        CUDA_TRY(ctx, cudaMemcpyAsync(out, ctx->gridQ.p, sizeof(float) * G3, cudaMemcpyDeviceToDevice, ctx->stream));
    } else {
        CUDA_TRY(ctx, cudaMemcpyAsync(out, ctx->grid.p, sizeof(float) * G3, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    return SQEQ_OK;
}
