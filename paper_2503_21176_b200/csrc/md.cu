// md.cu -- a-11: shadow XL-BOMD step driver (Eqs. 19-27; DESIGN.md R-MD).
//
// One time level needs (md_eval):
//   1. v = ke*phi[n] and the per-unit-charge field f[n]            -- Coulomb evaluation #1
//   2. q[n], lambda from the quasi-diagonal system Eq. 22 (closed form, two reductions)
//   3. f[q-n]                                                       -- Coulomb evaluation #2
//      F_i = ke (q_i f[n]_i + n_i f[q-n]_i) = -grad_i of Eq. 20's 1/2 (2q-n)' Phi n at fixed q, n
//      (bilinear form: -grad_i a'Phi b = a_i f[b]_i + b_i f[a]_i), plus the harmonic stand-in for
//      V_short (Eq. 14)
//   4. dt^2 ndd from Eq. 27, J x = -kappa (q[n]-n), by `krylov_rank` GMRES steps from zero; each
//      J w = -w - (ke phi[w] + dlambda)/u (Eq. 24 applied to Eq. 22) is one potential-only
//      Coulomb evaluation                                           -- evaluations #3 .. #2+m
// and a step is velocity Verlet for R around one md_eval, with
//   n(t+dt) = 2 n(t) - n(t-dt) + dt^2 ndd(t) + alpha_diss sum_k c_k n(t-k dt).
// All per-atom work runs in the kernels below; fp64 for n, q and every reduction.
#include <math.h>

#include "common.cuh"

#define ACC_CONV 0.00964853321   // (eV/Angstrom)/amu -> Angstrom/fs^2

// scal[] slots used here (0 and 1 belong to assemble / influence)
enum { S_T = 2, S_INVU = 3, S_U = 4, S_RES2 = 5, S_JAC = 6, S_EKIN = 7, S_VSTAND = 8 };

__device__ __forceinline__ void block_sum_to(double v, double* dst)
{
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 8) {
        v = red[threadIdx.x];
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) v += __shfl_xor_sync(0xffu, v, o);
        if (threadIdx.x == 0) atomicAdd(dst, v);
    }
    __syncthreads();
}

// v += dt/2 * a ; optionally x += dt * v ; optionally accumulate the kinetic energy (eV)
__global__ void __launch_bounds__(256)
k_md_kick(int64_t n, float* __restrict__ pos, float* __restrict__ vel, const float* __restrict__ force,
          const float* __restrict__ mass, double dt, int drift, double* __restrict__ ekin)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double ek = 0.0;
    if (i < n) {
        const double m = (double)mass[i];
        const double s = 0.5 * dt * ACC_CONV / m;
        double v2 = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double v = (double)vel[3 * i + d] + s * (double)force[3 * i + d];
            vel[3 * i + d] = (float)v;
            if (drift) pos[3 * i + d] = (float)((double)pos[3 * i + d] + dt * v);
            v2 += v * v;
        }
        ek = 0.5 * m * v2 / ACC_CONV;
    }
    if (ekin) block_sum_to(ek, ekin);
}

// Verlet step with dissipation for n; rows 0..5 = n(t-k dt), row 6 = dt^2 ndd(t)
struct NCoef { double a; double c[6]; };
__global__ void k_md_n_update(int64_t n, double* __restrict__ nh, NCoef k)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double v[6];
#pragma unroll
    for (int r = 0; r < 6; ++r) v[r] = nh[r * n + i];
    double d = 0.0;
#pragma unroll
    for (int r = 0; r < 6; ++r) d += k.c[r] * v[r];
    nh[i] = 2.0 * v[0] - v[1] + nh[6 * n + i] + k.a * d;
#pragma unroll
    for (int r = 1; r < 6; ++r) nh[r * n + i] = v[r - 1];
}

__global__ void k_md_hist_fill(int64_t n, const float* __restrict__ q0, double* __restrict__ nh)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = q0 ? (double)q0[i] : nh[i];
#pragma unroll
    for (int r = 0; r < 6; ++r) nh[r * n + i] = v;
}

// Eq. 22, first reduction: sum_i (chi_i + v_i)/u_i and sum_i 1/u_i
__global__ void __launch_bounds__(256)
k_md_q_pass1(int64_t n, const float* __restrict__ chi, const float* __restrict__ u,
             const float* __restrict__ phi, double ke, double* __restrict__ scal)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double t = 0.0, iu = 0.0;
    if (i < n) {
        iu = 1.0 / (double)u[i];
        t = ((double)chi[i] + ke * (double)phi[i]) * iu;
    }
    block_sum_to(t, scal + S_T);
    block_sum_to(iu, scal + S_INVU);
}

// Eq. 22 solved: lambda = -(Qtot + sum (chi+v)/u)/sum(1/u), q_i = -(chi_i + v_i + lambda)/u_i;
// residual d = q - n; shadow energy of Eq. 20: sum q chi + 1/2 q^2 u + (q - n/2) v
__global__ void __launch_bounds__(256)
k_md_q_pass2(int64_t n, const float* __restrict__ chi, const float* __restrict__ u,
             const float* __restrict__ phi, double ke, double qtot, const double* __restrict__ nv,
             double* __restrict__ q, double* __restrict__ d, double* __restrict__ scal)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const double lam = -(qtot + scal[S_T]) / scal[S_INVU];
    double e = 0.0, r2 = 0.0;
    if (i < n) {
        const double v = ke * (double)phi[i], c = (double)chi[i], uu = (double)u[i], ni = nv[i];
        const double qi = -(c + v + lam) / uu;
        q[i] = qi;
        d[i] = qi - ni;
        e = qi * c + 0.5 * qi * qi * uu + (qi - 0.5 * ni) * v;
        r2 = (qi - ni) * (qi - ni);
    }
    block_sum_to(e, scal + S_U);
    block_sum_to(r2, scal + S_RES2);
}

__global__ void k_md_forces(int64_t n, const double* __restrict__ q, const double* __restrict__ nv,
                            const float* __restrict__ fn, const float* __restrict__ fd, double ke,
                            float* __restrict__ force)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double qi = q[i], ni = nv[i];
#pragma unroll
    for (int k = 0; k < 3; ++k)
        force[3 * i + k] = (float)(ke * (qi * (double)fn[3 * i + k] + ni * (double)fd[3 * i + k]));
}

// harmonic stand-in for V_short: atoms 3m, 3m+1, 3m+2 = O, H, H (one thread per molecule)
__global__ void __launch_bounds__(256)
k_md_standin(int64_t nmol, const float* __restrict__ pos, double k_oh, double r_oh, double k_hh,
             double r_hh, float* __restrict__ force, double* __restrict__ vsum)
{
    int64_t m = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double V = 0.0;
    if (m < nmol) {
        double x[3][3], f[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int k = 0; k < 3; ++k) x[a][k] = (double)pos[9 * m + 3 * a + k];
        const int pa[3] = {0, 0, 1}, pb[3] = {1, 2, 2};
#pragma unroll
        for (int t = 0; t < 3; ++t) {
            const double kk = t < 2 ? k_oh : k_hh, r0 = t < 2 ? r_oh : r_hh;
            double dx[3], r2 = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) { dx[k] = x[pb[t]][k] - x[pa[t]][k]; r2 += dx[k] * dx[k]; }
            const double r = sqrt(r2);
            V += 0.5 * kk * (r - r0) * (r - r0);
            const double g = r > 0.0 ? kk * (r - r0) / r : 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) { f[pa[t]][k] += g * dx[k]; f[pb[t]][k] -= g * dx[k]; }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int k = 0; k < 3; ++k) force[9 * m + 3 * a + k] += (float)f[a][k];
    }
    if (vsum) block_sum_to(V, vsum);
}

// Eq. 24 applied to Eq. 22: (J w)_i = -w_i - (ke phi[w]_i + dlambda)/u_i, dlambda from sum(Jw + w) = 0
__global__ void __launch_bounds__(256)
k_md_jac_reduce(int64_t n, const float* __restrict__ u, const float* __restrict__ phi, double ke,
                double* __restrict__ scal)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double t = 0.0;
    if (i < n) t = ke * (double)phi[i] / (double)u[i];
    block_sum_to(t, scal + S_JAC);
}

__global__ void k_md_jac_apply(int64_t n, const double* __restrict__ w, const float* __restrict__ u,
                               const float* __restrict__ phi, double ke, const double* __restrict__ scal,
                               double* __restrict__ out)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double dl = -scal[S_JAC] / scal[S_INVU];
    out[i] = -w[i] - (ke * (double)phi[i] + dl) / (double)u[i];
}

__global__ void k_md_scale(int64_t n, double a, const double* __restrict__ x, double* __restrict__ y)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) y[i] = a * x[i];
}

// ------------------------------------------------------------------------------------------------
static int check_md_args(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3],
                         const sqeq_md_params* p, const char* who)
{
    if (!p) return sqeq_fail(ctx, SQEQ_EINVAL, "%s: params is NULL", who);
    SQEQ_TRY(validate_coulomb_args(ctx, nl, n, box, p->rc, p->alpha, p->grid, p->order, who));
    if (!(p->dt > 0.0) || !(p->ke > 0.0) || p->krylov_rank < 0 || p->krylov_rank > 64)
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: need dt > 0, ke > 0, 0 <= krylov_rank <= 64", who);
    if ((p->k_oh != 0.0 || p->k_hh != 0.0) && n % 3 != 0)
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: the O,H,H stand-in needs n divisible by 3", who);
    return SQEQ_OK;
}

// Forces F(R, n), dt^2 ndd and energies at one time level.  nhist row 0 = n, row 6 <- dt^2 ndd.
static int md_eval(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3],
                   const sqeq_md_params* p, const float* chi, const float* u, double* nhist,
                   float* force, int* evals)
{
    cudaStream_t st = ctx->stream;
    const int nb = ceil_div(n, 256);
    for (int k = 0; k < 2; ++k) SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_f[k], sizeof(float) * n));
    for (int k = 0; k < 2; ++k) SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_f3[k], sizeof(float) * 3 * n));
    for (int k = 0; k < 2; ++k) SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_d[k], sizeof(double) * n));
    float* phi = (float*)ctx->vec_f[0].p;
    float* phi_w = (float*)ctx->vec_f[1].p;
    float* f_n = (float*)ctx->vec_f3[0].p;
    float* f_d = (float*)ctx->vec_f3[1].p;
    double* q = (double*)ctx->vec_d[0].p;
    double* res = (double*)ctx->vec_d[1].p;
    double* scal = (double*)ctx->scal.p;
    double* nv = nhist;

    SQEQ_TRY(pme_setup(ctx, box, p->alpha, p->grid, p->order));
    SQEQ_TRY(prep_atoms(ctx, nl, pos, chi, ctx->K, st));            // geometry; charge slot set below
    SQEQ_TRY(prep_charges(ctx, nl, nullptr, nv, st));
    // all 2 + m evaluations of this time level share the geometry: the first one writes the cache (t and g)
    SQEQ_TRY(coulomb_eval(ctx, nl, n, box, p->rc, p->alpha, phi, f_n, false, true, GEOM_FIXED));
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        CUDA_TRY(ctx, cudaMemsetAsync(scal + S_T, 0, sizeof(double) * 7, st));
        k_md_q_pass1<<<nb, 256, 0, st>>>(n, chi, u, phi, p->ke, scal);
        KERNEL_CHECK(ctx);
        k_md_q_pass2<<<nb, 256, 0, st>>>(n, chi, u, phi, p->ke, p->total_charge, nv, q, res, scal);
        KERNEL_CHECK(ctx);
    }
    SQEQ_TRY(prep_charges(ctx, nl, nullptr, res, st));
    SQEQ_TRY(coulomb_eval(ctx, nl, n, box, p->rc, p->alpha, nullptr, f_d, false, true, GEOM_FIXED));     // field only
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        k_md_forces<<<nb, 256, 0, st>>>(n, q, nv, f_n, f_d, p->ke, force);
        KERNEL_CHECK(ctx);
        if (p->k_oh != 0.0 || p->k_hh != 0.0) {
            k_md_standin<<<ceil_div(n / 3, 256), 256, 0, st>>>(n / 3, pos, p->k_oh, p->r_oh, p->k_hh,
                                                                p->r_hh, force, scal + S_VSTAND);
            KERNEL_CHECK(ctx);
        }
    }
    int iters = 0;
    double* ndd = nhist + 6 * n;
    if (p->krylov_rank == 0) {
        // J ~ -I (the paper's remark that the solve may be loose): x = kappa (q[n]-n)
        k_md_scale<<<nb, 256, 0, st>>>(n, p->kappa, res, ndd);
        KERNEL_CHECK(ctx);
    } else {
        auto load_rhs = [&](double* w) {
            k_md_scale<<<nb, 256, 0, st>>>(n, -p->kappa, res, w);
            KERNEL_CHECK(ctx);
            return (int)SQEQ_OK;
        };
        auto apply = [&](const double* w, double* out) {
            SQEQ_TRY(prep_charges(ctx, nl, nullptr, w, st));
            SQEQ_TRY(coulomb_eval(ctx, nl, n, box, p->rc, p->alpha, phi_w, nullptr, false, false, GEOM_FIXED));
            StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
            CUDA_TRY(ctx, cudaMemsetAsync(scal + S_JAC, 0, sizeof(double), st));
            k_md_jac_reduce<<<nb, 256, 0, st>>>(n, u, phi_w, p->ke, scal);
            KERNEL_CHECK(ctx);
            k_md_jac_apply<<<nb, 256, 0, st>>>(n, w, u, phi_w, p->ke, scal, out);
            KERNEL_CHECK(ctx);
            return (int)SQEQ_OK;
        };
        double* x = nullptr;
        SQEQ_TRY(gmres_solve(ctx, n, apply, load_rhs, 0.0, p->krylov_rank, 0, &x, &iters, nullptr, nullptr));
        CUDA_TRY(ctx, cudaMemcpyAsync(ndd, x, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    }
    if (evals) *evals = 2 + iters;
    return SQEQ_OK;
}

static int md_read_energies(sqeq_ctx* ctx, double* energies, int evals)
{
    if (!energies) return SQEQ_OK;
    cudaStream_t st = ctx->stream;
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal.p, sizeof(double) * 9, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    energies[0] = ctx->h_scal[S_U] + ctx->h_scal[S_VSTAND];
    energies[1] = ctx->h_scal[S_EKIN];
    energies[2] = sqrt(ctx->h_scal[S_RES2]);
    energies[3] = (double)evals;
    return SQEQ_OK;
}

extern "C" int sqeq_shadow_md_init(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                                   const double box[3], const sqeq_md_params* p, const float* chi,
                                   const float* u, double tol, int max_iter, double* nhist, float* force,
                                   double* energies)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(check_md_args(ctx, nl, n, box, p, "sqeq_shadow_md_init"));
    if (!pos || !chi || !u || !nhist || !force)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_shadow_md_init: NULL argument");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    int solve_iters = 0;
    if (max_iter > 0) {
        // n(0) = q_min: Eq. 18 solved to `tol` (history start, DESIGN.md R-MD)
        SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_f[2], sizeof(float) * n));
        float* q0 = (float*)ctx->vec_f[2].p;
        SQEQ_TRY(sqeq_qeq_solve(ctx, nl, n, pos, box, p->rc, p->alpha, p->grid, p->order, p->ke, chi, u,
                                p->total_charge, tol, max_iter, 0, q0, nullptr, &solve_iters, nullptr));
        k_md_hist_fill<<<ceil_div(n, 256), 256, 0, st>>>(n, q0, nhist);
    } else {
        k_md_hist_fill<<<ceil_div(n, 256), 256, 0, st>>>(n, nullptr, nhist);   // rows 1..5 <- row 0
    }
    KERNEL_CHECK(ctx);
    int evals = 0;
    SQEQ_TRY(md_eval(ctx, nl, n, pos, box, p, chi, u, nhist, force, &evals));
    return md_read_energies(ctx, energies, evals + solve_iters);
}

extern "C" int sqeq_shadow_md_step(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, float* pos, float* vel,
                                   const float* mass, const double box[3], const sqeq_md_params* p,
                                   const float* chi, const float* u, double* nhist, float* force,
                                   double* energies)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(check_md_args(ctx, nl, n, box, p, "sqeq_shadow_md_step"));
    if (!pos || !vel || !mass || !chi || !u || !nhist || !force)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_shadow_md_step: NULL argument");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int nb = ceil_div(n, 256);
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        k_md_kick<<<nb, 256, 0, st>>>(n, pos, vel, force, mass, p->dt, 1, nullptr);
        KERNEL_CHECK(ctx);
        NCoef k;
        k.a = p->alpha_diss;
        for (int r = 0; r < 6; ++r) k.c[r] = p->c[r];
        k_md_n_update<<<nb, 256, 0, st>>>(n, nhist, k);
        KERNEL_CHECK(ctx);
    }
    int evals = 0;
    SQEQ_TRY(md_eval(ctx, nl, n, pos, box, p, chi, u, nhist, force, &evals));
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        k_md_kick<<<nb, 256, 0, st>>>(n, pos, vel, force, mass, p->dt, 0, (double*)ctx->scal.p + S_EKIN);
        KERNEL_CHECK(ctx);
    }
    return md_read_energies(ctx, energies, evals);
}
