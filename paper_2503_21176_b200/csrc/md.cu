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
#include <string.h>

#include "common.cuh"

#define ACC_CONV 0.00964853321   // (eV/Angstrom)/amu -> Angstrom/fs^2

// scal[] slots used here (0 and 1 belong to assemble / influence)
enum { S_T = 2, S_INVU = 3, S_U = 4, S_RES2 = 5, S_JAC = 6, S_EKIN = 7, S_VSTAND = 8 };   // 12: max drift (nlist.cu)

// blocks of exactly 256 threads
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

// V_short stand-in, second part: soft-sphere repulsion 1/2 k (r0 - r)^2 between oxygens (caller index 3m) of
// different molecules, r < r0.  One warp per atom of the list's cell-major order (non-oxygens leave at once); the
// warp sweeps the 27 cells around the atom's build-time cell -- r0 + skin <= cell edge, so every partner is there
// although the cells are those of the last build -- with the periodic image of each cell applied; each pair is
// seen from both sides, so only atom i is written (no atomics) and the energy is halved.
struct RepGeom {
    int nc[3];
    float L[3];
    float k, r0;
};
// The oxygens of the list's cell-major order, cell by cell (built once per list): counts per cell, a one-block scan,
// the fill.
__global__ void k_rep_count(int ncells, const int* __restrict__ cell_start, const int* __restrict__ perm, int* __restrict__ ostart)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncells) return;
    int m = 0;
    for (int t = cell_start[c]; t < cell_start[c + 1]; ++t) m += perm[t] % 3 == 0;
    ostart[c] = m;
}
__global__ void __launch_bounds__(1024) k_rep_scan(int ncells, int* __restrict__ ostart)     // exclusive, in place; [ncells] = total
{
    __shared__ int s_w[32];
    __shared__ int s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int b = 0; b < ncells; b += 1024) {
        const int c = b + threadIdx.x;
        const int v = c < ncells ? ostart[c] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) s_w[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int w = s_w[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += y;
            }
            s_w[lane] = w;
        }
        __syncthreads();
        const int carry = s_carry, before = wid ? s_w[wid - 1] : 0;
        if (c < ncells) ostart[c] = carry + before + x - v;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = carry + s_w[31];
        __syncthreads();
    }
    if (threadIdx.x == 0) ostart[ncells] = s_carry;
}
__global__ void k_rep_fill(int ncells, const int* __restrict__ cell_start, const int* __restrict__ perm,
                           const int* __restrict__ ostart, int* __restrict__ oslot)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncells) return;
    int o = ostart[c];
    for (int t = cell_start[c]; t < cell_start[c + 1]; ++t)
        if (perm[t] % 3 == 0) oslot[o++] = t;
}

// One THREAD per oxygen, in cell order (the lanes of a warp sit in the same or neighbouring cells, so their candidate
// loads mostly coincide).  An oxygen visits only the neighbouring cells it can reach: along an axis the cell below
// (above) is needed when the atom lies within `reach` = r0 + skin of its cell's lower (upper) face -- positions are the
// current ones on the build-time image, and both atoms of a pair have moved at most skin/2 since the cells were filled
// (check_md_args: reach <= cell edge): on average 12 of the 27 cells, 5 oxygens each.  (One warp per atom over all
// atoms of all 27 cells took 0.73 ms at 331,776 atoms.)
__global__ void __launch_bounds__(256)
k_md_oo_repulsion(int no, const float4* __restrict__ xq, const int* __restrict__ cell_of, const int* __restrict__ ostart,
                  const int* __restrict__ oslot, const int* __restrict__ perm, RepGeom g, float reach,
                  float* __restrict__ force, double* __restrict__ vsum)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    double V = 0.0;
    if (k < no) {
        const int s = oslot[k];
        const float4 xi = xq[s];
        const int c = cell_of[s];
        const int cc[3] = {c & 1023, (c >> 10) & 1023, c >> 20};
        const float xs[3] = {xi.x, xi.y, xi.z};
        int lo[3], hi[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const float edge = g.L[d] / (float)g.nc[d], off = xs[d] - (float)cc[d] * edge;
            lo[d] = off < reach ? -1 : 0;
            hi[d] = edge - off < reach ? 1 : 0;
        }
        const float r02 = g.r0 * g.r0;
        float fx = 0.f, fy = 0.f, fz = 0.f, v = 0.f;
        for (int dx = lo[0]; dx <= hi[0]; ++dx)
            for (int dy = lo[1]; dy <= hi[1]; ++dy)
                for (int dz = lo[2]; dz <= hi[2]; ++dz) {
                    int ux = cc[0] + dx, uy = cc[1] + dy, uz = cc[2] + dz;
                    float sx = 0.f, sy = 0.f, sz = 0.f;
                    if (ux < 0) { ux += g.nc[0]; sx = -g.L[0]; } else if (ux >= g.nc[0]) { ux -= g.nc[0]; sx = g.L[0]; }
                    if (uy < 0) { uy += g.nc[1]; sy = -g.L[1]; } else if (uy >= g.nc[1]) { uy -= g.nc[1]; sy = g.L[1]; }
                    if (uz < 0) { uz += g.nc[2]; sz = -g.L[2]; } else if (uz >= g.nc[2]) { uz -= g.nc[2]; sz = g.L[2]; }
                    const int cell = (ux * g.nc[1] + uy) * g.nc[2] + uz;
                    const int beg = ostart[cell], end = ostart[cell + 1];
                    for (int t = beg; t < end; ++t) {
                        const float4 xj = xq[oslot[t]];
                        const float ddx = xi.x - (xj.x + sx), ddy = xi.y - (xj.y + sy), ddz = xi.z - (xj.z + sz);
                        const float r2 = ddx * ddx + ddy * ddy + ddz * ddz;
                        if (r2 < r02 && r2 > 0.f) {                           // r2 = 0: the atom itself (zero image)
                            const float r = sqrtf(r2);
                            const float f = g.k * (g.r0 - r) / r;
                            fx += f * ddx; fy += f * ddy; fz += f * ddz;
                            v += 0.25f * g.k * (g.r0 - r) * (g.r0 - r);        // half of the pair energy
                        }
                    }
                }
        const int64_t oi = perm[s];
        force[3 * oi + 0] += fx;
        force[3 * oi + 1] += fy;
        force[3 * oi + 2] += fz;
        V = (double)v;
    }
    if (vsum) block_sum_to(V, vsum);
}

// The oxygen lists of the stand-in repulsion belong to the neighbour list: built once per list.  The step entries
// call this BEFORE a CUDA-graph capture (workspace growth synchronises, and the three kernels need not be replayed).
static int standin_prepare(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const sqeq_md_params* p, cudaStream_t st)
{
    if (p->k_rep == 0.0 || (ctx->rep_nl == nl && ctx->rep_serial == nl->serial)) return SQEQ_OK;
    const int ncells = nl->ncell[0] * nl->ncell[1] * nl->ncell[2], no = (int)(n / 3);
    SQEQ_TRY(sqeq_reserve(ctx, ctx->rep_oslot, sizeof(int) * (size_t)(no + 1)));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->rep_ostart, sizeof(int) * (size_t)(ncells + 1)));
    k_rep_count<<<ceil_div(ncells, 256), 256, 0, st>>>(ncells, nl->cell_start, nl->perm, (int*)ctx->rep_ostart.p);
    k_rep_scan<<<1, 1024, 0, st>>>(ncells, (int*)ctx->rep_ostart.p);
    k_rep_fill<<<ceil_div(ncells, 256), 256, 0, st>>>(ncells, nl->cell_start, nl->perm, (const int*)ctx->rep_ostart.p,
                                                    (int*)ctx->rep_oslot.p);
    ctx->launches += 2;
    KERNEL_CHECK(ctx);
    ctx->rep_nl = nl;
    ctx->rep_serial = nl->serial;
    return SQEQ_OK;
}

// both parts of the stand-in, added to `force`; V into scal[S_VSTAND]
static int standin_run(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const sqeq_md_params* p,
                       float* force, cudaStream_t st)
{
    double* scal = (double*)ctx->scal.p;
    if (p->k_oh != 0.0 || p->k_hh != 0.0) {
        k_md_standin<<<ceil_div(n / 3, 256), 256, 0, st>>>(n / 3, pos, p->k_oh, p->r_oh, p->k_hh, p->r_hh, force,
                                                            scal + S_VSTAND);
        KERNEL_CHECK(ctx);
    }
    if (p->k_rep != 0.0) {
        RepGeom g;
        for (int d = 0; d < 3; ++d) { g.nc[d] = nl->ncell[d]; g.L[d] = (float)nl->box[d]; }
        g.k = (float)p->k_rep; g.r0 = (float)p->r_rep;
        const float reach = (float)(p->r_rep + (nl->cutoff - p->rc)) * 1.0001f;
        const int ncells = nl->ncell[0] * nl->ncell[1] * nl->ncell[2], no = (int)(n / 3);
        SQEQ_TRY(standin_prepare(ctx, nl, n, p, st));       // no-op when the step entry already did it (outside a capture)
        k_md_oo_repulsion<<<ceil_div(no, 256), 256, 0, st>>>(no, (const float4*)ctx->xq.p, nl->cell_of, (const int*)ctx->rep_ostart.p,
                                                            (const int*)ctx->rep_oslot.p, nl->perm, g, reach, force,
                                                            scal + S_VSTAND);
        KERNEL_CHECK(ctx);
    }
    return SQEQ_OK;
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
    if ((p->k_oh != 0.0 || p->k_hh != 0.0 || p->k_rep != 0.0) && n % 3 != 0)
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: the O,H,H stand-in needs n divisible by 3", who);
    if (!(p->krylov_tol >= 0.0)) return sqeq_fail(ctx, SQEQ_EINVAL, "%s: krylov_tol must be >= 0", who);
    if (p->k_rep != 0.0) {
        double edge = 1e300;
        for (int d = 0; d < 3; ++d) edge = fmin(edge, nl->box[d] / nl->ncell[d]);
        if (!(p->r_rep > 0.0) || p->r_rep + (nl->cutoff - p->rc) > edge)
            return sqeq_fail(ctx, SQEQ_EINVAL, "%s: r_rep = %g plus the skin %g must not exceed the list's cell edge %g",
                             who, p->r_rep, nl->cutoff - p->rc, edge);
    }
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
        SQEQ_TRY(standin_run(ctx, nl, n, pos, p, force, st));
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
        SQEQ_TRY(gmres_solve(ctx, n, apply, load_rhs, p->krylov_tol, p->krylov_rank, 0, &x, &iters, nullptr, nullptr));
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

// one step, enqueued: half kick + drift, n update, md_eval at the new time level, second half kick
static int md_step_enqueue(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, float* pos, float* vel, const float* mass,
                           const double box[3], const sqeq_md_params* p, const float* chi, const float* u,
                           double* nhist, float* force, int* evals)
{
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
    SQEQ_TRY(md_eval(ctx, nl, n, pos, box, p, chi, u, nhist, force, evals));
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        k_md_kick<<<nb, 256, 0, st>>>(n, pos, vel, force, mass, p->dt, 0, (double*)ctx->scal.p + S_EKIN);
        KERNEL_CHECK(ctx);
    }
    return SQEQ_OK;
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
    int evals = 0;
    SQEQ_TRY(md_step_enqueue(ctx, nl, n, pos, vel, mass, box, p, chi, u, nhist, force, &evals));
    return md_read_energies(ctx, energies, evals);
}

// nsteps steps with the neighbour list kept valid by the library (rebuilt when the largest displacement
// since the build exceeds half the skin).  The host must not wait for the GPU every step, so the test runs two steps
// behind: after step s the displacement the atoms will have two position updates later, |x + 2 dt v - x0|, is
// reduced on the device and copied to pinned memory; before step s + 2 the host looks at that number (the GPU is
// long past it) and rebuilds if it reaches skin/2 - slack (slack covers the 2 dt^2 a the extrapolation leaves out).
// The first two steps after a (re)build, for which no such number exists yet, are checked synchronously.
extern "C" int sqeq_shadow_md_run(sqeq_ctx* ctx, sqeq_nlist** nl_io, int64_t n, float* pos, float* vel,
                                  const float* mass, const double box[3], const sqeq_md_params* p, const float* chi,
                                  const float* u, double* nhist, float* force, int nsteps, double list_cutoff,
                                  double slack, double* stats)
{
    if (!ctx) return SQEQ_EINVAL;
    if (!nl_io || !*nl_io) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_shadow_md_run: needs a list built for the current positions");
    SQEQ_TRY(check_md_args(ctx, *nl_io, n, box, p, "sqeq_shadow_md_run"));
    if (!pos || !vel || !mass || !chi || !u || !nhist || !force || nsteps < 1)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_shadow_md_run: NULL argument or nsteps < 1");
    const double half_skin = 0.5 * (list_cutoff - p->rc);
    if (!(list_cutoff == (*nl_io)->cutoff) || !(slack >= 0.0) || !(half_skin - slack > 0.0))
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_shadow_md_run: list_cutoff must be the list's cutoff and skin/2 > slack >= 0");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    if (!ctx->d_ring) {
        CUDA_TRY(ctx, cudaMalloc((void**)&ctx->d_ring, 4 * sizeof(unsigned)));
        CUDA_TRY(ctx, cudaMallocHost((void**)&ctx->h_ring, 4 * sizeof(unsigned)));
        for (auto& e : ctx->ring_ev) CUDA_TRY(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    uint64_t ring_serial[4] = {0, 0, 0, 0};
    int rebuilds = 0, evals = 0;
    double worst_ahead = 0.0;
    auto rebuild = [&]() -> int {
        sqeq_nlist* fresh = nullptr;
        SQEQ_TRY(nl_build_impl(ctx, n, pos, box, list_cutoff, &fresh));
        nl_release(*nl_io);
        *nl_io = fresh;
        ++rebuilds;
        return SQEQ_OK;
    };
    for (int s = 0; s < nsteps; ++s) {
        sqeq_nlist* nl = *nl_io;
        double ahead = -1.0;
        if (s >= 2 && ring_serial[(s - 2) & 3] == nl->serial) {
            CUDA_TRY(ctx, cudaEventSynchronize(ctx->ring_ev[(s - 2) & 3]));
            float d2;
            memcpy(&d2, &ctx->h_ring[(s - 2) & 3], sizeof(float));
            ahead = sqrt((double)d2);
        } else {
            SQEQ_TRY(nl_max_drift_impl(ctx, nl, pos, vel, p->dt, &ahead));      // synchronous, one update ahead
        }
        if (ahead > worst_ahead && ahead < half_skin - slack) worst_ahead = ahead;
        if (!(ahead < half_skin - slack)) SQEQ_TRY(rebuild());
        nl = *nl_io;
        {
            // every step on one list is the same ~120 launches: a CUDA graph, re-captured (and updated in place)
            // after a rebuild
            uint64_t key = hash_mix(0x3d, nl->serial);
            for (uint64_t v : {(uint64_t)(uintptr_t)pos, (uint64_t)(uintptr_t)vel, (uint64_t)(uintptr_t)mass, (uint64_t)(uintptr_t)chi,
                               (uint64_t)(uintptr_t)u, (uint64_t)(uintptr_t)nhist, (uint64_t)(uintptr_t)force, (uint64_t)n})
                key = hash_mix(key, v);
            const unsigned char* pb = (const unsigned char*)p;
            for (size_t k = 0; k < sizeof(sqeq_md_params); ++k) key = hash_mix(key, pb[k]);
            SQEQ_TRY(standin_prepare(ctx, nl, n, p, st));
            SQEQ_TRY(graph_run(ctx, 1, key, [&]() { return md_step_enqueue(ctx, nl, n, pos, vel, mass, box, p, chi, u, nhist, force, &evals); }));
            ctx->gc.valid = false;          // replays move the atoms without passing through prep_atoms on the host
            ctx->geom_serial++;
        }
        unsigned* d = ctx->d_ring + (s & 3);
        SQEQ_TRY(nl_max_drift_enqueue(ctx, nl, pos, vel, 2.0 * p->dt, d));
        CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_ring + (s & 3), d, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(ctx, cudaEventRecord(ctx->ring_ev[s & 3], st));
        ring_serial[s & 3] = nl->serial;
    }
    double en[4] = {0, 0, 0, 0};
    SQEQ_TRY(md_read_energies(ctx, en, evals));
    double drift_now = 0.0;
    SQEQ_TRY(nl_max_drift_impl(ctx, *nl_io, pos, nullptr, 0.0, &drift_now));
    if (stats) {
        stats[0] = en[0]; stats[1] = en[1]; stats[2] = en[2]; stats[3] = en[3];
        stats[4] = (double)rebuilds; stats[5] = worst_ahead; stats[6] = drift_now; stats[7] = half_skin;
    }
    return SQEQ_OK;
}

// ------------------------------------------------------------------------------------------------
// Regular Born-Oppenheimer MD (NEXT-2): q_min by GMRES on Eq. 18, forces at fixed q_min.
__global__ void __launch_bounds__(256)
k_bomd_energy(int64_t n, const double* __restrict__ q, const float* __restrict__ chi, const float* __restrict__ u,
              double* __restrict__ out)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double e = 0.0;
    if (i < n) e = q[i] * (double)chi[i] + 0.5 * q[i] * q[i] * (double)u[i];
    block_sum_to(e, out);
}

__global__ void k_bomd_scale_force(int64_t n3, float ke, float* __restrict__ f)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n3) f[i] *= ke;
}

static int bomd_eval(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3],
                     const sqeq_md_params* p, const float* chi, const float* u, double tol, int max_iter, bool jacobi,
                     bool warm, double* q, double* lambda, float* force, double* energies, double ekin_scalar_ready)
{
    (void)ekin_scalar_ready;
    cudaStream_t st = ctx->stream;
    const int nb = ceil_div(n, 256);
    double* scal = (double*)ctx->scal.p;
    SQEQ_TRY(pme_setup(ctx, box, p->alpha, p->grid, p->order));
    SQEQ_TRY(prep_atoms(ctx, nl, pos, nullptr, ctx->K, st));
    int iters = 0;
    double relres = 1.0;
    bool converged = false;
    SQEQ_TRY(qeq_solve_prepared(ctx, nl, n, box, p->rc, p->alpha, p->ke, chi, u, p->total_charge, tol, max_iter, 0,
                                jacobi, warm, q, lambda, &iters, &relres, &converged));
    // forces at fixed q = q_min (Eq. 19) and E_Coul[q] on the same geometry (the cache the solve left behind)
    SQEQ_TRY(sqeq_reserve(ctx, ctx->vec_f[1], sizeof(float) * n));
    SQEQ_TRY(prep_charges(ctx, nl, nullptr, q, st));
    SQEQ_TRY(coulomb_eval(ctx, nl, n, box, p->rc, p->alpha, (float*)ctx->vec_f[1].p, force, true, false, GEOM_FIXED));
    {
        StageTimer tm(ctx, SQEQ_T_KRYLOV, st);
        CUDA_TRY(ctx, cudaMemsetAsync(scal + S_U, 0, sizeof(double), st));
        CUDA_TRY(ctx, cudaMemsetAsync(scal + S_VSTAND, 0, sizeof(double), st));
        k_bomd_energy<<<nb, 256, 0, st>>>(n, q, chi, u, scal + S_U);
        KERNEL_CHECK(ctx);
        k_bomd_scale_force<<<ceil_div(3 * n, 256), 256, 0, st>>>(3 * n, (float)p->ke, force);
        KERNEL_CHECK(ctx);
        SQEQ_TRY(standin_run(ctx, nl, n, pos, p, force, st));
    }
    if (energies) { energies[2] = relres; energies[3] = (double)(iters + 1); }
    return converged ? SQEQ_OK : SQEQ_ENOTCONV;
}

static int bomd_read(sqeq_ctx* ctx, const sqeq_md_params* p, double* energies)
{
    cudaStream_t st = ctx->stream;
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal.p, sizeof(double) * 9, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if (energies) {
        energies[0] = ctx->h_scal[S_U] + p->ke * ctx->h_scal[0] + ctx->h_scal[S_VSTAND];    // scal[0]: E_Coul (k_e = 1)
        energies[1] = ctx->h_scal[S_EKIN];
    }
    return SQEQ_OK;
}

extern "C" int sqeq_bomd_init(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3],
                              const sqeq_md_params* p, const float* chi, const float* u, double tol, int max_iter,
                              int jacobi, double* q, double* lambda, float* force, double* energies)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(check_md_args(ctx, nl, n, box, p, "sqeq_bomd_init"));
    if (!pos || !chi || !u || !q || !lambda || !force || max_iter < 1 || !(tol >= 0.0))
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_bomd_init: NULL argument, max_iter < 1 or tol < 0");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaMemsetAsync((double*)ctx->scal.p + S_EKIN, 0, sizeof(double), ctx->stream));
    const int r = bomd_eval(ctx, nl, n, pos, box, p, chi, u, tol, max_iter, jacobi != 0, false, q, lambda, force, energies, 0);
    if (r != SQEQ_OK && r != SQEQ_ENOTCONV) return r;
    SQEQ_TRY(bomd_read(ctx, p, energies));
    if (r == SQEQ_ENOTCONV) return sqeq_fail(ctx, SQEQ_ENOTCONV, "sqeq_bomd_init: tol %.3e not reached in %d evaluations", tol, max_iter);
    return SQEQ_OK;
}

extern "C" int sqeq_bomd_step(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, float* pos, float* vel, const float* mass,
                              const double box[3], const sqeq_md_params* p, const float* chi, const float* u, double tol,
                              int max_iter, int jacobi, int warm_start, double* q, double* lambda, float* force,
                              double* energies)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(check_md_args(ctx, nl, n, box, p, "sqeq_bomd_step"));
    if (!pos || !vel || !mass || !chi || !u || !q || !lambda || !force || max_iter < 1 || !(tol >= 0.0))
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_bomd_step: NULL argument, max_iter < 1 or tol < 0");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int nb = ceil_div(n, 256);
    k_md_kick<<<nb, 256, 0, st>>>(n, pos, vel, force, mass, p->dt, 1, nullptr);
    KERNEL_CHECK(ctx);
    const int r = bomd_eval(ctx, nl, n, pos, box, p, chi, u, tol, max_iter, jacobi != 0, warm_start != 0, q, lambda, force, energies, 0);
    if (r != SQEQ_OK && r != SQEQ_ENOTCONV) return r;
    CUDA_TRY(ctx, cudaMemsetAsync((double*)ctx->scal.p + S_EKIN, 0, sizeof(double), st));
    k_md_kick<<<nb, 256, 0, st>>>(n, pos, vel, force, mass, p->dt, 0, (double*)ctx->scal.p + S_EKIN);
    KERNEL_CHECK(ctx);
    SQEQ_TRY(bomd_read(ctx, p, energies));
    if (r == SQEQ_ENOTCONV) return sqeq_fail(ctx, SQEQ_ENOTCONV, "sqeq_bomd_step: tol %.3e not reached in %d evaluations", tol, max_iter);
    return SQEQ_OK;
}
