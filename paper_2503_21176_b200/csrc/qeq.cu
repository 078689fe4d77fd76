// qeq.cu -- a-10: matrix-free GMRES on the QEq KKT system, Eq. 18:
//     [ C  1 ] [ q      ]   [ -chi ]
//     [ 1' 0 ] [ lambda ] = [ Qtot ],     C v = J o v + ke * phi[v]
// Each Krylov iteration is one potential-only Coulomb evaluation on fixed geometry ("Each
// iteration involves calculating a Coulomb-like potential").  Krylov basis, dots and
// updates are fp64 on the device; the (m+1) x m Hessenberg least-squares problem (Givens
// rotations) is solved on the host.  Orthogonalisation: classical Gram-Schmidt applied twice
// (CGS2), which needs two batched dot/update launches per iteration instead of j sequential ones.
// Zero initial guess, no preconditioner (DESIGN.md R-G13).
#include <math.h>

#include <functional>
#include <vector>

#include "common.cuh"

int validate_coulomb_args(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3],
                          double rc, double alpha, const int grid[3], int order, const char* who);

// b = [-chi ; Qtot]  -> V0 (unnormalised), also accumulates ||b||^2 into nrm2
__global__ void k_qeq_rhs(int64_t n, const float* __restrict__ chi, double qtot, double* __restrict__ v0)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) v0[i] = -(double)chi[i];
    else if (i == n) v0[n] = qtot;
}

// w = A v for v = [v_q ; mu]:  w_i = J_i v_i + ke phi_i + mu,  w_N = sum_i v_i (accumulated atomically)
__global__ void k_qeq_matvec(int64_t n, const double* __restrict__ v, const float* __restrict__ J,
                             const float* __restrict__ phi, double ke, double* __restrict__ w)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double s = 0.0;
    if (i < n) {
        const double vi = v[i];
        w[i] = (double)J[i] * vi + ke * (double)phi[i] + v[n];
        s = vi;
    }
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 8) {
        s = red[threadIdx.x];
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) s += __shfl_xor_sync(0xffu, s, o);
        if (threadIdx.x == 0) atomicAdd(w + n, s);
    }
}

// h[k] += <V_k, w> for k < nv; grid = (chunks, nv); V has leading dimension ld
#define DOT_CHUNK 2048
__global__ void __launch_bounds__(256)
k_dots(int64_t len, int64_t ld, const double* __restrict__ V, const double* __restrict__ w,
       double* __restrict__ h)
{
    const double* vk = V + (int64_t)blockIdx.y * ld;
    const int64_t beg = (int64_t)blockIdx.x * DOT_CHUNK;
    const int64_t end = beg + DOT_CHUNK < len ? beg + DOT_CHUNK : len;
    double s = 0.0;
    for (int64_t i = beg + threadIdx.x; i < end; i += 256) s += vk[i] * w[i];
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 8) {
        s = red[threadIdx.x];
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) s += __shfl_xor_sync(0xffu, s, o);
        if (threadIdx.x == 0) atomicAdd(h + blockIdx.y, s);
    }
}

// w -= sum_k h[k] V_k
__global__ void k_sub_combo(int64_t len, int64_t ld, int nv, const double* __restrict__ V,
                            const double* __restrict__ h, double* __restrict__ w)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= len) return;
    // eight loads in flight per thread: with one accumulator the loop runs at the latency of its load (2.4 TB/s at 25
    // vectors of 331,777 doubles)
    double a0 = w[i], a1 = 0.0, a2 = 0.0, a3 = 0.0;
    const double* v = V + i;
    int k = 0;
    for (; k + 8 <= nv; k += 8) {
        double x[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = v[(int64_t)(k + j) * ld];
        a0 -= h[k] * x[0]; a1 -= h[k + 1] * x[1]; a2 -= h[k + 2] * x[2]; a3 -= h[k + 3] * x[3];
        a0 -= h[k + 4] * x[4]; a1 -= h[k + 5] * x[5]; a2 -= h[k + 6] * x[6]; a3 -= h[k + 7] * x[7];
    }
    for (; k < nv; ++k) a0 -= h[k] * v[(int64_t)k * ld];
    w[i] = (a0 + a1) + (a2 + a3);
}

// Fused steps of the twice-applied classical Gram-Schmidt sweep.  A dot product is a sum over chunks, and an element of
// the updated w depends on that element only, so the block that updates a chunk can form the chunk's share of the NEXT
// reduction in the same pass:
//   k_sub_dots<NV>: w -= sum_k h[k] V_k, then h2[k] += <V_k, w> over the chunk   (nv <= NV basis vectors in registers)
//   k_sub_norm:     w -= sum_k h[k] V_k, then nrm2 += <w, w> over the chunk      (any nv)
// One pass over V and one launch less each than k_sub_combo followed by k_dots.
template <int NV>
__global__ void __launch_bounds__(256)
k_sub_dots(int64_t len, int64_t ld, int nv, const double* __restrict__ V, const double* __restrict__ h,
           double* __restrict__ w, double* __restrict__ h2)
{
    const int64_t beg = (int64_t)blockIdx.x * DOT_CHUNK;
    const int64_t end = beg + DOT_CHUNK < len ? beg + DOT_CHUNK : len;
    double hk[NV], s[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) { hk[k] = k < nv ? h[k] : 0.0; s[k] = 0.0; }
    for (int64_t i = beg + threadIdx.x; i < end; i += 256) {
        double v[NV], acc = w[i];
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            v[k] = k < nv ? V[(int64_t)k * ld + i] : 0.0;
            acc -= hk[k] * v[k];
        }
        w[i] = acc;
#pragma unroll
        for (int k = 0; k < NV; ++k) s[k] += v[k] * acc;
    }
    __shared__ double red[NV][8];
#pragma unroll
    for (int k = 0; k < NV; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
        if ((threadIdx.x & 31) == 0) red[k][threadIdx.x >> 5] = s[k];
    }
    __syncthreads();
    if (threadIdx.x < 8 * NV) {
        const int k = threadIdx.x >> 3;
        double t = red[k][threadIdx.x & 7];
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o, 8);
        if ((threadIdx.x & 7) == 0 && k < nv) atomicAdd(h2 + k, t);
    }
}

__global__ void __launch_bounds__(256)
k_sub_norm(int64_t len, int64_t ld, int nv, const double* __restrict__ V, const double* __restrict__ h,
           double* __restrict__ w, double* __restrict__ nrm2)
{
    const int64_t beg = (int64_t)blockIdx.x * DOT_CHUNK;
    const int64_t end = beg + DOT_CHUNK < len ? beg + DOT_CHUNK : len;
    double s = 0.0;
    for (int64_t i = beg + threadIdx.x; i < end; i += 256) {
        double acc = w[i];
        for (int k = 0; k < nv; ++k) acc -= h[k] * V[(int64_t)k * ld + i];
        w[i] = acc;
        s += acc * acc;
    }
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 8) {
        s = red[threadIdx.x];
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) s += __shfl_xor_sync(0xffu, s, o);
        if (threadIdx.x == 0) atomicAdd(nrm2, s);
    }
}

// The sweep for column j: h = V^T w, w -= V h, h2 = V^T w, w -= V h2, nrm2 = |w|^2 (h, h2, nrm2 zeroed by the caller).
static void cgs2_sweep(sqeq_ctx* ctx, int64_t len, int64_t ld, int nv, const double* V, double* w, double* h, double* h2,
                       double* nrm2, cudaStream_t st)
{
    ctx->launches += nv <= 8 ? 2 : 4;                       // the caller's KERNEL_CHECK counts the last one
    const int nchunk = ceil_div(len, DOT_CHUNK), nbl = ceil_div(len, 256);
    k_dots<<<dim3(nchunk, nv), 256, 0, st>>>(len, ld, V, w, h);
    if (nv <= 8) {
        // short bases (the rank-m updates of shadow MD, the first columns of a solve): launch-bound, fused
        if (nv <= 4) k_sub_dots<4><<<nchunk, 256, 0, st>>>(len, ld, nv, V, h, w, h2);
        else k_sub_dots<8><<<nchunk, 256, 0, st>>>(len, ld, nv, V, h, w, h2);
        k_sub_norm<<<nchunk, 256, 0, st>>>(len, ld, nv, V, h2, w, nrm2);
    } else {
        // long bases: bandwidth-bound passes over V, which want one thread per element (measured at 50 vectors:
        // 0.482 ms per iteration fused, 0.452 this way)
        k_sub_combo<<<nbl, 256, 0, st>>>(len, ld, nv, V, h, w);
        k_dots<<<dim3(nchunk, nv), 256, 0, st>>>(len, ld, V, w, h2);
        k_sub_combo<<<nbl, 256, 0, st>>>(len, ld, nv, V, h2, w);
        k_dots<<<dim3(nchunk, 1), 256, 0, st>>>(len, ld, w, w, nrm2);
    }
}

// x += sum_k y[k] V_k
__global__ void k_add_combo(int64_t len, int64_t ld, int nv, const double* __restrict__ V,
                            const double* __restrict__ y, double* __restrict__ x)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= len) return;
    double acc = x[i];
    for (int k = 0; k < nv; ++k) acc += y[k] * V[(int64_t)k * ld + i];
    x[i] = acc;
}

// dst = src * (1/sqrt(*nrm2))
__global__ void k_normalise(int64_t len, const double* __restrict__ src, const double* __restrict__ nrm2,
                            double* __restrict__ dst)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= len) return;
    const double s = *nrm2 > 0.0 ? rsqrt(*nrm2) : 0.0;
    dst[i] = src[i] * s;
}

__global__ void k_axpby(int64_t len, double a, const double* __restrict__ x, double b, double* __restrict__ y)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < len) y[i] = a * x[i] + b * y[i];
}

// z = x o d (right Jacobi preconditioner: d holds the inverse diagonal)
__global__ void k_hadamard(int64_t len, const double* __restrict__ x, const double* __restrict__ d, double* __restrict__ z)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < len) z[i] = x[i] * d[i];
}

// x += d o sum_k y[k] V_k
__global__ void k_add_combo_scaled(int64_t len, int64_t ld, int nv, const double* __restrict__ V,
                                   const double* __restrict__ y, const double* __restrict__ d, double* __restrict__ x)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= len) return;
    double acc = 0.0;
    for (int k = 0; k < nv; ++k) acc += y[k] * V[(int64_t)k * ld + i];
    x[i] += d[i] * acc;
}

// inverse diagonal of Eq. 18's matrix: 1/(J_i + ke A_ii) on the charge rows, 1 on the constraint row
__global__ void k_qeq_jacobi(int64_t n, const float* __restrict__ J, double keAii, double* __restrict__ dinv)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) dinv[i] = 1.0 / ((double)J[i] + keAii);
    else if (i == n) dinv[n] = 1.0;
}

// x0 = [q0 ; lambda0]
__global__ void k_qeq_guess(int64_t n, const double* __restrict__ q0, double lam0, double* __restrict__ x)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) x[i] = q0[i];
    else if (i == n) x[n] = lam0;
}

__global__ void k_d2f(int64_t n, const double* __restrict__ x, float* __restrict__ y)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) y[i] = (float)x[i];
}

__global__ void k_f2d(int64_t n, const float* __restrict__ x, double* __restrict__ y)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) y[i] = (double)x[i];
}

// ------------------------------------------------------------------------------------------------
// Generic GMRES on device fp64 vectors of length `len` (leading dimension ld).  Zero initial guess.
//   apply(v, w): w = A v        load_rhs(w): w = b
// On return x (ctx->kry_w + ld) holds the iterate.  Host side: Givens-rotated Hessenberg.
// Least-squares problem of a finished GMRES cycle, on the device (one thread: m <= 64 columns of a few numbers):
// Hessenberg columns from the CGS2 coefficients of each iteration (hcols[j]: first pass [m+2], second pass [m+2],
// |w|^2), Givens rotations, back substitution.  y[0..m) <- the combination coefficients (0 beyond an exact
// breakdown), *relres <- the residual estimate |g_k| / |b|.  scratch: (m+1) m + 3 m + 1 doubles.
__global__ void k_gmres_lsq(int m, const double* __restrict__ hcols, const double* __restrict__ bn2,
                            double* __restrict__ scratch, double* __restrict__ y, double* __restrict__ relres)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int HL = 2 * (m + 2) + 1;
    double* H = scratch;
    double* cs = H + (size_t)(m + 1) * m;
    double* sn = cs + m;
    double* g = sn + m;
    const double bnorm = sqrt(*bn2);
    for (int k = 0; k <= m; ++k) g[k] = 0.0;
    g[0] = bnorm;
    int kd = m;
    for (int j = 0; j < m; ++j) {
        const double* hc = hcols + (size_t)j * HL;
        double* Hj = H + (size_t)j * (m + 1);
        for (int k = 0; k <= j; ++k) Hj[k] = hc[k] + hc[(m + 2) + k];
        Hj[j + 1] = sqrt(hc[2 * (m + 2)]);
        for (int k = 0; k < j; ++k) {
            const double t = cs[k] * Hj[k] + sn[k] * Hj[k + 1];
            Hj[k + 1] = -sn[k] * Hj[k] + cs[k] * Hj[k + 1];
            Hj[k] = t;
        }
        const double a = Hj[j], b = Hj[j + 1], rr = hypot(a, b);
        cs[j] = rr > 0 ? a / rr : 1.0;
        sn[j] = rr > 0 ? b / rr : 0.0;
        Hj[j] = rr;
        Hj[j + 1] = 0.0;
        g[j + 1] = -sn[j] * g[j];
        g[j] = cs[j] * g[j];
        if (b == 0.0) { kd = j + 1; break; }
    }
    for (int i = 0; i < m; ++i) y[i] = 0.0;
    for (int i = kd - 1; i >= 0; --i) {
        double sacc = g[i];
        for (int l = i + 1; l < kd; ++l) sacc -= H[(size_t)l * (m + 1) + i] * y[l];
        const double d = H[(size_t)i * (m + 1) + i];
        y[i] = d != 0.0 ? sacc / d : 0.0;
    }
    *relres = bnorm > 0.0 ? fabs(g[kd]) / bnorm : 0.0;
}

// m GMRES iterations from a zero initial guess with NO host synchronisation (the rank-m updates of Eq. 27, timed
// Krylov loops): coefficients stay on the device, k_gmres_lsq solves the small problem there.  relres_host may be
// NULL (then the call returns with everything merely enqueued -- a whole MD step can be captured in a CUDA graph).
static int gmres_fixed_async(sqeq_ctx* ctx, int64_t len, const std::function<int(const double*, double*)>& apply,
                             const std::function<int(double*)>& load_rhs, int m, double** x_out, double* relres_host,
                             const double* dinv)
{
    cudaStream_t st = ctx->stream;
    const int64_t ld = (len + 31) & ~(int64_t)31;
    const size_t HL = (size_t)2 * (m + 2) + 1;
    const size_t nh = HL * m + 1 + m + 1 + (size_t)(m + 1) * m + 3 * m + 1;
    SQEQ_TRY(sqeq_reserve(ctx, ctx->kry_V, sizeof(double) * (size_t)ld * (m + 1)));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->kry_w, sizeof(double) * (size_t)ld * 3));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->kry_h, sizeof(double) * nh));
    double* V = (double*)ctx->kry_V.p;
    double* w = (double*)ctx->kry_w.p;
    double* x = w + ld;
    double* z = w + 2 * ld;
    double* hcols = (double*)ctx->kry_h.p;
    double* bn2 = hcols + HL * m;
    double* y = bn2 + 1;
    double* relres = y + m;
    double* scratch = relres + 1;
    const int nbl = ceil_div(len, 256);
    const int nchunk = ceil_div(len, DOT_CHUNK);
    *x_out = x;
    SQEQ_TRY(load_rhs(w));
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        CUDA_TRY(ctx, cudaMemsetAsync(hcols, 0, sizeof(double) * (HL * m + 1), st));       // all coefficients and |b|^2
        CUDA_TRY(ctx, cudaMemsetAsync(x, 0, sizeof(double) * ld, st));
        k_dots<<<dim3(nchunk, 1), 256, 0, st>>>(len, ld, w, w, bn2);
        KERNEL_CHECK(ctx);
        k_normalise<<<nbl, 256, 0, st>>>(len, w, bn2, V);
        KERNEL_CHECK(ctx);
    }
    for (int j = 0; j < m; ++j) {
        if (dinv) {
            k_hadamard<<<nbl, 256, 0, st>>>(len, V + (int64_t)j * ld, dinv, z);
            KERNEL_CHECK(ctx);
            SQEQ_TRY(apply(z, w));
        } else {
            SQEQ_TRY(apply(V + (int64_t)j * ld, w));
        }
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        double* h = hcols + HL * j;
        double* h2 = h + (m + 2);
        double* nrm2 = h2 + (m + 2);
        cgs2_sweep(ctx, len, ld, j + 1, V, w, h, h2, nrm2, st);
        KERNEL_CHECK(ctx);
        k_normalise<<<nbl, 256, 0, st>>>(len, w, nrm2, V + (int64_t)(j + 1) * ld);
        KERNEL_CHECK(ctx);
    }
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        k_gmres_lsq<<<1, 32, 0, st>>>(m, hcols, bn2, scratch, y, relres);
        KERNEL_CHECK(ctx);
        if (dinv) k_add_combo_scaled<<<nbl, 256, 0, st>>>(len, ld, m, V, y, dinv, x);
        else k_add_combo<<<nbl, 256, 0, st>>>(len, ld, m, V, y, x);
        KERNEL_CHECK(ctx);
    }
    if (relres_host) {
        CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal + 4, relres, sizeof(double), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(ctx, cudaStreamSynchronize(st));
        *relres_host = ctx->h_scal[4];
    }
    return SQEQ_OK;
}

// x0 (device, may be NULL): initial guess; its residual b - A x0 costs one operator application.
// dinv (device, may be NULL): right Jacobi preconditioner, the solve runs on A D^-1 y = b with x = D^-1 y
// ("Jacobi preconditioner is used for regular MD runs").
int gmres_solve(sqeq_ctx* ctx, int64_t len, const std::function<int(const double*, double*)>& apply,
                const std::function<int(double*)>& load_rhs, double tol, int max_iter, int restart,
                double** x_out, int* iters_out, double* relres_out, bool* converged_out,
                const double* x0, const double* dinv)
{
    cudaStream_t st = ctx->stream;
    const int m = restart > 0 ? (restart < max_iter ? restart : max_iter) : max_iter;
    if (tol <= 0.0 && !x0 && m == max_iter && m <= 64) {
        // a fixed number of iterations in one cycle: nothing for the host to decide, nothing to wait for
        if (iters_out) *iters_out = m;
        if (converged_out) *converged_out = false;
        return gmres_fixed_async(ctx, len, apply, load_rhs, m, x_out, relres_out, dinv);
    }
    const int64_t ld = (len + 31) & ~(int64_t)31;
    SQEQ_TRY(sqeq_reserve(ctx, ctx->kry_V, sizeof(double) * (size_t)ld * (m + 1)));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->kry_w, sizeof(double) * (size_t)ld * 3));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->kry_h, sizeof(double) * (size_t)(2 * (m + 2) + 2)));
    double* V = (double*)ctx->kry_V.p;
    double* w = (double*)ctx->kry_w.p;
    double* x = w + ld;
    double* z = w + 2 * ld;                      // D^-1 v_j
    double* h = (double*)ctx->kry_h.p;          // [m+2] first-pass coefficients
    double* h2 = h + (m + 2);                    // second pass
    double* nrm2 = h2 + (m + 2);
    const int nbl = ceil_div(len, 256);
    const int nchunk = ceil_div(len, DOT_CHUNK);
    if (x0) CUDA_TRY(ctx, cudaMemcpyAsync(x, x0, sizeof(double) * len, cudaMemcpyDeviceToDevice, st));
    else CUDA_TRY(ctx, cudaMemsetAsync(x, 0, sizeof(double) * ld, st));
    *x_out = x;

    // |b|
    double bnorm = 0.0;
    {
        SQEQ_TRY(load_rhs(w));
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        CUDA_TRY(ctx, cudaMemsetAsync(nrm2, 0, sizeof(double), st));
        k_dots<<<dim3(nchunk, 1), 256, 0, st>>>(len, ld, w, w, nrm2);
        KERNEL_CHECK(ctx);
        CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal + 4, nrm2, sizeof(double), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(ctx, cudaStreamSynchronize(st));
        bnorm = sqrt(ctx->h_scal[4]);
    }
    int iters = 0;
    double relres = 1.0;
    bool converged = false;
    if (bnorm == 0.0) { converged = true; relres = 0.0; }
    bool first_cycle = x0 == nullptr;       // with a guess the first cycle starts from r = b - A x0, like a restart
    std::vector<double> H((size_t)(m + 1) * m), cs(m), sn(m), gvec(m + 1), y(m);
    // Column j of the Hessenberg matrix from the coefficients of iteration j (hc), its Givens rotation and the
    // residual estimate; true when the cycle ends at this column (converged or exact breakdown).
    const size_t HL = (size_t)2 * (m + 2) + 1;
    auto process_column = [&](int j, const double* hc) {
        double* Hj = H.data() + (size_t)j * (m + 1);
        for (int k = 0; k <= j; ++k) Hj[k] = hc[k] + hc[(m + 2) + k];
        Hj[j + 1] = sqrt(hc[2 * (m + 2)]);
        for (int k = 0; k < j; ++k) {
            double t = cs[k] * Hj[k] + sn[k] * Hj[k + 1];
            Hj[k + 1] = -sn[k] * Hj[k] + cs[k] * Hj[k + 1];
            Hj[k] = t;
        }
        double a = Hj[j], b = Hj[j + 1], rr = hypot(a, b);
        cs[j] = rr > 0 ? a / rr : 1.0;
        sn[j] = rr > 0 ? b / rr : 0.0;
        Hj[j] = rr;
        Hj[j + 1] = 0.0;
        gvec[j + 1] = -sn[j] * gvec[j];
        gvec[j] = cs[j] * gvec[j];
        relres = fabs(gvec[j + 1]) / bnorm;
        if (relres <= tol || b == 0.0) { converged = relres <= tol; return true; }
        return false;
    };
    // tol <= 0 asks for a FIXED number of iterations (the rank-m updates of Eq. 27, timed Krylov loops): the
    // host has nothing to decide between iterations, so the coefficients of every iteration are copied to
    // pinned memory without synchronising and the columns are processed after the cycle -- the GPU never
    // waits for the host to launch the next iteration.
    // tol > 0: the host must see every column, but not before the next iteration is launched: the coefficients go to
    // pinned memory with an event behind them and column j is judged while iteration j + 1 runs (LAG = 1; 2 was no
    // faster).  When the tolerance is met at column j the solution is formed from columns 0..j; the one application
    // already launched beyond it is wasted work, not counted in *iters_out, and cheaper than idling the GPU for a host
    // round trip every iteration (tolerance 1e-5 at cfg 4: 0.49 -> 0.44 ms per iteration, cfg 2: 0.16 -> 0.135).
    const bool deferred = tol <= 0.0;
    constexpr int LAG = 1;
    if (!ctx->kry_ev[0])
        for (auto& e : ctx->kry_ev) CUDA_TRY(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    if (ctx->h_kry_cap < HL * (size_t)m) {
        if (ctx->h_kry) cudaFreeHost(ctx->h_kry);
        ctx->h_kry = nullptr;
        ctx->h_kry_cap = 0;
        CUDA_TRY(ctx, cudaMallocHost((void**)&ctx->h_kry, sizeof(double) * HL * (size_t)m));
        ctx->h_kry_cap = HL * (size_t)m;
    }
    while (!converged && iters < max_iter) {
        // r = b - A x  (x = 0 in the first cycle: r = b, already in w)
        double beta = bnorm;
        if (!first_cycle) {
            double* r = V;  // reuse V_0 as scratch for A x
            SQEQ_TRY(apply(x, r));
            ++iters;
            SQEQ_TRY(load_rhs(w));
            StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
            k_axpby<<<nbl, 256, 0, st>>>(len, -1.0, r, 1.0, w);
            KERNEL_CHECK(ctx);
            CUDA_TRY(ctx, cudaMemsetAsync(nrm2, 0, sizeof(double), st));
            k_dots<<<dim3(nchunk, 1), 256, 0, st>>>(len, ld, w, w, nrm2);
            KERNEL_CHECK(ctx);
            CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal + 4, nrm2, sizeof(double), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(ctx, cudaStreamSynchronize(st));
            beta = sqrt(ctx->h_scal[4]);
            relres = beta / bnorm;
            if (relres <= tol) { converged = true; break; }
        }
        first_cycle = false;
        {
            StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
            k_normalise<<<nbl, 256, 0, st>>>(len, w, nrm2, V);
            KERNEL_CHECK(ctx);
        }
        std::fill(gvec.begin(), gvec.end(), 0.0);
        gvec[0] = beta;
        int j = 0, judged = 0;
        bool ended = false;
        for (; j < m && iters < max_iter; ++j) {
            if (dinv) {
                k_hadamard<<<nbl, 256, 0, st>>>(len, V + (int64_t)j * ld, dinv, z);
                KERNEL_CHECK(ctx);
                SQEQ_TRY(apply(z, w));
            } else {
                SQEQ_TRY(apply(V + (int64_t)j * ld, w));
            }
            ++iters;
            {
                StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
                CUDA_TRY(ctx, cudaMemsetAsync(h, 0, sizeof(double) * (2 * (m + 2) + 1), st));
                cgs2_sweep(ctx, len, ld, j + 1, V, w, h, h2, nrm2, st);
                KERNEL_CHECK(ctx);
                k_normalise<<<nbl, 256, 0, st>>>(len, w, nrm2, V + (int64_t)(j + 1) * ld);
                KERNEL_CHECK(ctx);
                CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_kry + HL * (size_t)j, h, sizeof(double) * HL, cudaMemcpyDeviceToHost, st));
                if (!deferred) CUDA_TRY(ctx, cudaEventRecord(ctx->kry_ev[j & 3], st));
            }
            if (!deferred && j >= LAG) {
                CUDA_TRY(ctx, cudaEventSynchronize(ctx->kry_ev[(j - LAG) & 3]));
                if (process_column(j - LAG, ctx->h_kry + HL * (size_t)(j - LAG))) { ended = true; ++j; break; }
                ++judged;
            }
        }
        {
            // the columns not judged yet: all of them (fixed count), or the last LAG of a cycle that ran out
            const int launched = j;
            if (ended) {
                j = judged + 1;                          // columns 0..judged make the solution
                iters -= launched - j;                   // look-ahead applications beyond it
            } else {
                if (deferred) CUDA_TRY(ctx, cudaStreamSynchronize(st));
                for (j = judged; j < launched; ++j) {
                    if (!deferred) CUDA_TRY(ctx, cudaEventSynchronize(ctx->kry_ev[j & 3]));
                    if (process_column(j, ctx->h_kry + HL * (size_t)j)) { ++j; break; }     // converged / exact breakdown
                }
                iters -= launched - j;
            }
        }
        // y = R^{-1} g ;  x += V y
        const int k = j;
        for (int i = k - 1; i >= 0; --i) {
            double s = gvec[i];
            for (int l = i + 1; l < k; ++l) s -= H[(size_t)l * (m + 1) + i] * y[l];
            y[i] = s / H[(size_t)i * (m + 1) + i];
        }
        if (k > 0) {
            StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
            CUDA_TRY(ctx, cudaMemcpyAsync(h, y.data(), sizeof(double) * k, cudaMemcpyHostToDevice, st));
            if (dinv) k_add_combo_scaled<<<nbl, 256, 0, st>>>(len, ld, k, V, h, dinv, x);
            else k_add_combo<<<nbl, 256, 0, st>>>(len, ld, k, V, h, x);
            KERNEL_CHECK(ctx);
            CUDA_TRY(ctx, cudaStreamSynchronize(st));   // y is a host vector reused next cycle
        }
        if (converged || restart == 0) break;
    }
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = relres;
    if (converged_out) *converged_out = converged;
    return SQEQ_OK;
}

// w = A v for Eq. 18 (one potential-only Coulomb evaluation on the prepared geometry)
struct QeqOp {
    sqeq_ctx* ctx;
    const sqeq_nlist* nl;
    int64_t n;
    const double* box;
    double rc, alpha, ke;
    const float* J;
    float* phi;   // scratch [n]
};

static int qeq_apply_body(const QeqOp& op, const double* v, double* w)
{
    sqeq_ctx* ctx = op.ctx;
    cudaStream_t st = ctx->stream;
    const int64_t n = op.n;
    SQEQ_TRY(prep_charges(ctx, op.nl, nullptr, v, st));
    // fixed geometry: the first mat-vec writes the geometry cache, the others are sparse products over it
    SQEQ_TRY(coulomb_eval(ctx, op.nl, n, op.box, op.rc, op.alpha, op.phi, nullptr, false, false, GEOM_FIXED));
    StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
    CUDA_TRY(ctx, cudaMemsetAsync(w + n, 0, sizeof(double), st));
    k_qeq_matvec<<<ceil_div(n, 256), 256, 0, st>>>(n, v, op.J, op.phi, op.ke, w);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

static int qeq_apply(const QeqOp& op, const double* v, double* w)
{
    sqeq_ctx* ctx = op.ctx;
    cudaStream_t st = ctx->stream;
    const int64_t n = op.n;
    const sqeq_nlist* nl = op.nl;
    // Small systems are launch-bound (648 atoms: a dozen kernels of ~3 us per mat-vec against ~6 us of host time per
    // launch).  Once the geometry cache is warm every mat-vec is the same sequence of launches: the Krylov vector is
    // copied into a fixed buffer, so that the arguments never change, and the sequence is replayed as a CUDA graph.
    const GeomCache& gc = ctx->gc;
    const bool warm = gc.valid && gc.nl == nl && gc.serial == nl->serial && gc.rc == op.rc && gc.alpha == op.alpha && nl->fmt == 1;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (n > 65536 || !warm || !ctx->graphs || ctx->profiling || st == nullptr || st == cudaStreamLegacy ||
        cudaStreamIsCapturing(st, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone)
        return qeq_apply_body(op, v, w);
    SQEQ_TRY(sqeq_reserve(ctx, ctx->qeq_vin, sizeof(double) * (size_t)(n + 1)));
    double* vin = (double*)ctx->qeq_vin.p;
    CUDA_TRY(ctx, cudaMemcpyAsync(vin, v, sizeof(double) * (size_t)(n + 1), cudaMemcpyDeviceToDevice, st));
    uint64_t key = hash_mix(0x53, nl->serial);
    double kd[3] = {op.rc, op.alpha, op.ke};
    uint64_t kb[3];
    memcpy(kb, kd, sizeof(kb));
    for (uint64_t x : {(uint64_t)(uintptr_t)nl, (uint64_t)(uintptr_t)vin, (uint64_t)(uintptr_t)w, (uint64_t)(uintptr_t)op.phi,
                       (uint64_t)(uintptr_t)op.J, (uint64_t)n, kb[0], kb[1], kb[2], (uint64_t)ctx->K[0], (uint64_t)ctx->K[1],
                       (uint64_t)ctx->K[2], (uint64_t)ctx->order})
        key = hash_mix(key, x);
    return graph_run(ctx, 2, key, [&]() { return qeq_apply_body(op, vin, w); });
}

// A_ii of the Ewald matrix for r_c < L/2 (no image of an atom inside its own cutoff): the reciprocal-space self
// term (1/(pi V)) sum_{m != 0} exp(-pi^2 |m/L|^2/alpha^2)/|m/L|^2 minus 2 alpha/sqrt(pi) (Eqs. 4-5)
double ewald_self_diag(const double box[3], double alpha)
{
    const double V = box[0] * box[1] * box[2];
    int mmax[3];
    for (int d = 0; d < 3; ++d) mmax[d] = (int)ceil(6.3 * alpha * box[d] / M_PI);     // exp(-39.7) ~ 6e-18
    // one octant with the multiplicity of its mirror images (the summand is even in each index)
    double s = 0.0;
    for (int a = 0; a <= mmax[0]; ++a)
        for (int b = 0; b <= mmax[1]; ++b)
            for (int c = 0; c <= mmax[2]; ++c) {
                if (!(a | b | c)) continue;
                const double m2 = (a / box[0]) * (a / box[0]) + (b / box[1]) * (b / box[1]) + (c / box[2]) * (c / box[2]);
                const double e = -M_PI * M_PI * m2 / (alpha * alpha);
                if (e < -40.0) break;                                   // the rest of this c row is smaller still
                s += (double)((a ? 2 : 1) * (b ? 2 : 1) * (c ? 2 : 1)) * exp(e) / m2;
            }
    return s / (M_PI * V) - 2.0 * alpha / sqrt(M_PI);
}

// Eq. 18 on prepared geometry: q (fp64 device [n], out; also the initial guess when warm != 0) and lambda.
int qeq_solve_prepared(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3], double rc, double alpha,
                       double ke, const float* chi, const float* J, double total_charge, double tol, int max_iter,
                       int restart, bool jacobi, bool warm, double* q_io, double* lambda_io, int* iters_out,
                       double* relres_out, bool* converged_out)
{
    cudaStream_t st = ctx->stream;
    const int64_t len = n + 1;
    const int nbl = ceil_div(len, 256);
    SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_f[0], sizeof(float) * n));
    QeqOp op{ctx, nl, n, box, rc, alpha, ke, J, (float*)ctx->vec_f[0].p};
    auto apply = [&](const double* v, double* w) { return qeq_apply(op, v, w); };
    auto load_rhs = [&](double* w) {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        k_qeq_rhs<<<nbl, 256, 0, st>>>(n, chi, total_charge, w);
        KERNEL_CHECK(ctx);
        return (int)SQEQ_OK;
    };
    double* dinv = nullptr;
    double* x0 = nullptr;
    if (jacobi || warm) {
        SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_d[4], sizeof(double) * len));
        SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_d[5], sizeof(double) * len));
    }
    if (jacobi) {
        dinv = (double*)ctx->vec_d[4].p;
        // the lattice sum behind A_ii (millions of terms at 150 A) once per (box, alpha), not once per solve: regular
        // BOMD solves every step (it was 75 of the 90 ms of a step at 331,776 atoms)
        if (!(ctx->diag_alpha == alpha && ctx->diag_box[0] == box[0] && ctx->diag_box[1] == box[1] && ctx->diag_box[2] == box[2])) {
            ctx->diag_val = ewald_self_diag(box, alpha);
            ctx->diag_alpha = alpha;
            for (int d = 0; d < 3; ++d) ctx->diag_box[d] = box[d];
        }
        k_qeq_jacobi<<<nbl, 256, 0, st>>>(n, J, ke * ctx->diag_val, dinv);
        KERNEL_CHECK(ctx);
    }
    if (warm) {
        x0 = (double*)ctx->vec_d[5].p;
        k_qeq_guess<<<nbl, 256, 0, st>>>(n, q_io, *lambda_io, x0);
        KERNEL_CHECK(ctx);
    }
    double* x = nullptr;
    SQEQ_TRY(gmres_solve(ctx, len, apply, load_rhs, tol, max_iter, restart, &x, iters_out, relres_out, converged_out, x0, dinv));
    CUDA_TRY(ctx, cudaMemcpyAsync(q_io, x, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal + 5, x + n, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    *lambda_io = ctx->h_scal[5];
    return SQEQ_OK;
}

static int qeq_solve_common(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3],
                            double rc, double alpha, const int grid[3], int order, double ke, const float* chi,
                            const float* J, double total_charge, double tol, int max_iter, int restart, bool jacobi,
                            const float* q0, double lambda0, float* q_out, double* lambda_out, int* iters_out,
                            double* relres_out, const char* who)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(validate_coulomb_args(ctx, nl, n, box, rc, alpha, grid, order, who));
    if (!pos || !chi || !J || !q_out) return sqeq_fail(ctx, SQEQ_EINVAL, "%s: NULL argument", who);
    if (max_iter < 1 || restart < 0 || !(tol >= 0.0))
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: need max_iter >= 1, restart >= 0, tol >= 0", who);
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    SQEQ_TRY(pme_setup(ctx, box, alpha, grid, order));
    // geometry once; the charge slot is refreshed per mat-vec
    SQEQ_TRY(prep_atoms(ctx, nl, pos, nullptr, ctx->K, st));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_d[3], sizeof(double) * (n + 1)));
    double* qd = (double*)ctx->vec_d[3].p;
    double lam = lambda0;
    if (q0) {
        k_f2d<<<ceil_div(n, 256), 256, 0, st>>>(n, q0, qd);
        KERNEL_CHECK(ctx);
    }
    int iters = 0;
    double relres = 1.0;
    bool converged = false;
    SQEQ_TRY(qeq_solve_prepared(ctx, nl, n, box, rc, alpha, ke, chi, J, total_charge, tol, max_iter, restart, jacobi,
                                q0 != nullptr, qd, &lam, &iters, &relres, &converged));
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        k_d2f<<<ceil_div(n, 256), 256, 0, st>>>(n, qd, q_out);
        KERNEL_CHECK(ctx);
        CUDA_TRY(ctx, cudaStreamSynchronize(st));
    }
    if (lambda_out) *lambda_out = lam;
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = relres;
    if (!converged)
        return sqeq_fail(ctx, SQEQ_ENOTCONV, "%s: relative residual %.3e > tol %.3e after %d Coulomb evaluations",
                         who, relres, tol, iters);
    return SQEQ_OK;
}

extern "C" int sqeq_qeq_solve(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                              const double box[3], double rc, double alpha, const int grid[3], int order,
                              double ke, const float* chi, const float* J, double total_charge,
                              double tol, int max_iter, int restart, float* q_out, double* lambda_out,
                              int* iters_out, double* relres_out)
{
    return qeq_solve_common(ctx, nl, n, pos, box, rc, alpha, grid, order, ke, chi, J, total_charge, tol, max_iter,
                            restart, false, nullptr, 0.0, q_out, lambda_out, iters_out, relres_out, "sqeq_qeq_solve");
}

extern "C" int sqeq_qeq_solve_pc(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                                 const double box[3], double rc, double alpha, const int grid[3], int order,
                                 double ke, const float* chi, const float* J, double total_charge,
                                 double tol, int max_iter, int restart, int jacobi, const float* q0, double lambda0,
                                 float* q_out, double* lambda_out, int* iters_out, double* relres_out)
{
    return qeq_solve_common(ctx, nl, n, pos, box, rc, alpha, grid, order, ke, chi, J, total_charge, tol, max_iter,
                            restart, jacobi != 0, q0, lambda0, q_out, lambda_out, iters_out, relres_out, "sqeq_qeq_solve_pc");
}
