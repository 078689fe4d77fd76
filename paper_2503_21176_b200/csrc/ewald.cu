// ewald.cu -- regular (direct) Ewald reciprocal sum, PAPER.md:98-132 (section 3.2, Eqs. 6-12), SURVEY.md 8(f) NEXT-3:
// the paper's second method, faster than PME below about 5,000 atoms, with the phase matrix
// M_ij = r_i . k_j of Eq. 9 never stored: it is formed block by block in shared memory / registers.
//
//   S(k)      = sum_i q_i e^{i k.r_i}                                           (Eqs. 7-9)
//   phi_i     = (4 pi/V) sum_k v_k [cos(k.r_i) Re S + sin(k.r_i) Im S]          (Eq. 11)
//   dE/dr_i   = (4 pi/V) sum_k v_k k q_i [cos(k.r_i) Im S - sin(k.r_i) Re S]    (Eq. 10 with the G2 reading of Eq. 12)
//   E_rec     = (2 pi/V) sum_k v_k |S(k)|^2,  v_k = exp(-k^2/4 alpha^2)/k^2     (Eq. 6 with the G1 reading)
// over all k = 2 pi (m_x/L_x, m_y/L_y, m_z/L_z), m != 0, |m_d| <= kmax_d.  Only the half space m_x >= 0 is visited
// (S(-k) = conj S(k)): weight 2 for m_x > 0, 1 in the plane m_x = 0 (which holds both k and -k).
//
// e^{i k.r} factorises per axis, so three per-atom tables e^{2 pi i m f_d} (f = fractional coordinate, formed in fp64
// from the raw caller position) are computed once; pass 1 (one thread per k-vector, atoms staged in shared memory
// chunk by chunk) multiplies three table entries per (atom, k); pass 2 (one thread per atom, coefficients w v S
// staged in shared memory) walks m_z by a phase recurrence restarted from the tables at every (m_x, m_y) row.
// Everything else of the evaluation -- real-space sum over the list, self term, assembly -- is the PME path's.
#include <math.h>

#include "common.cuh"

struct EwaldGeom {
    int kx, ky, kz;          // kmax per axis
    int ny, nz;              // 2 ky + 1, 2 kz + 1
    int ntab;                // (kx + 1) + ny + nz table rows
    int nk;                  // (kx + 1) ny nz half-space vectors
    double L[3];
    float four_pi_over_V;
    float kfac[3];           // 2 pi / L_d
};

// E[t][s]: t < kx+1: e^{2 pi i t f_x}; then m_y = -ky..ky; then m_z = -kz..kz.  s = cell-major (list) order.
__global__ void k_ewald_tables(int64_t n, const float* __restrict__ pos, const int* __restrict__ perm, EwaldGeom g,
                               float2* __restrict__ E)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int t = blockIdx.y;
    if (s >= n) return;
    int d, m;
    if (t <= g.kx) { d = 0; m = t; }
    else if (t < g.kx + 1 + g.ny) { d = 1; m = t - (g.kx + 1) - g.ky; }
    else { d = 2; m = t - (g.kx + 1) - g.ny - g.kz; }
    const double f = (double)pos[3 * (int64_t)perm[s] + d] / g.L[d];
    double a = (double)m * (f - floor(f));          // phase / 2 pi
    a -= floor(a);
    double sn, cs;
    sincospi(2.0 * a, &sn, &cs);
    E[(int64_t)t * n + s] = make_float2((float)cs, (float)sn);
}

// pass 1: structure factors, one thread per half-space k-vector
#define EW_CHUNK 32
__global__ void __launch_bounds__(256)
k_ewald_sf(int64_t n, const float2* __restrict__ E, const float4* __restrict__ xq, EwaldGeom g, float2* __restrict__ S)
{
    extern __shared__ float2 tab[];                 // [EW_CHUNK][ntab + 1] (row padded: consecutive m_z, distinct banks)
    __shared__ float qs[EW_CHUNK];
    const int ik = blockIdx.x * blockDim.x + threadIdx.x;
    const bool on = ik < g.nk;
    const int ikc = on ? ik : 0;
    const int mz = ikc % g.nz, my = (ikc / g.nz) % g.ny, mx = ikc / (g.nz * g.ny);
    const int tx = mx, ty = g.kx + 1 + my, tz = g.kx + 1 + g.ny + mz;
    const int row = g.ntab + 1;
    float sre = 0.f, sim = 0.f;
    for (int64_t i0 = 0; i0 < n; i0 += EW_CHUNK) {
        const int na = (int)min((int64_t)EW_CHUNK, n - i0);
        __syncthreads();
        for (int e = threadIdx.x; e < g.ntab * EW_CHUNK; e += blockDim.x) {
            const int t = e / EW_CHUNK, a = e % EW_CHUNK;       // consecutive threads: consecutive atoms (coalesced)
            if (a < na) tab[a * row + t] = E[(int64_t)t * n + i0 + a];
        }
        if (threadIdx.x < na) qs[threadIdx.x] = xq[i0 + threadIdx.x].w;
        __syncthreads();
        for (int a = 0; a < na; ++a) {
            const float2 ex = tab[a * row + tx], ey = tab[a * row + ty], ez = tab[a * row + tz];
            const float q = qs[a];
            const float pr = ex.x * ey.x - ex.y * ey.y, pi = ex.x * ey.y + ex.y * ey.x;
            sre = fmaf(q, pr * ez.x - pi * ez.y, sre);
            sim = fmaf(q, pr * ez.y + pi * ez.x, sim);
        }
    }
    if (on) S[ik] = make_float2(sre, sim);
}

// coefficients c_k = w v_k S(k) in place, E_rec = (2 pi/V) sum_half w v |S|^2 in fp64
__global__ void __launch_bounds__(256)
k_ewald_coef(EwaldGeom g, double alpha, float2* __restrict__ S, double* __restrict__ e_out)
{
    const int ik = blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (ik < g.nk) {
        const int mz = ik % g.nz - g.kz, my = (ik / g.nz) % g.ny - g.ky, mx = ik / (g.nz * g.ny);
        float2 s = S[ik];
        double w = 0.0;
        if (mx | my | mz) {
            const double kxv = 2.0 * M_PI * mx / g.L[0], kyv = 2.0 * M_PI * my / g.L[1], kzv = 2.0 * M_PI * mz / g.L[2];
            const double k2 = kxv * kxv + kyv * kyv + kzv * kzv;
            w = (mx > 0 ? 2.0 : 1.0) * exp(-k2 / (4.0 * alpha * alpha)) / k2;
        }
        e = w * ((double)s.x * s.x + (double)s.y * s.y);
        S[ik] = make_float2((float)(w * s.x), (float)(w * s.y));
    }
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x < 8) {
        e = red[threadIdx.x];
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) e += __shfl_xor_sync(0xffu, e, o);
        if (threadIdx.x == 0 && e_out) atomicAdd(e_out, 2.0 * M_PI / (g.L[0] * g.L[1] * g.L[2]) * e);
    }
}

// pass 2: potential and per-unit-charge field, one thread per atom; the coefficients of one m_x plane at a time
// in shared memory (every thread reads the same entry: a broadcast)
template <bool FORCE>
__global__ void __launch_bounds__(128)
k_ewald_gather(int64_t n, const float2* __restrict__ E, const float2* __restrict__ C, EwaldGeom g, float4* __restrict__ out)
{
    extern __shared__ float2 cs[];                  // [ny * nz]
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool on = s < n;
    const int64_t sc = on ? s : 0;
    const float2 ezmin = E[(int64_t)(g.kx + 1 + g.ny) * n + sc];          // m_z = -kz
    const float2 ezstep = E[(int64_t)(g.kx + 1 + g.ny + g.kz + 1) * n + sc];   // m_z = +1 (kz >= 1)
    float ph = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
    const int plane = g.ny * g.nz;
    for (int mx = 0; mx <= g.kx; ++mx) {
        __syncthreads();
        for (int e = threadIdx.x; e < plane; e += blockDim.x) cs[e] = C[mx * plane + e];
        __syncthreads();
        const float2 ex = E[(int64_t)mx * n + sc];
        for (int iy = 0; iy < g.ny; ++iy) {
            const float2 ey = E[(int64_t)(g.kx + 1 + iy) * n + sc];
            const float xr = ex.x * ey.x - ex.y * ey.y, xi = ex.x * ey.y + ex.y * ey.x;
            float pr = xr * ezmin.x - xi * ezmin.y, pi = xr * ezmin.y + xi * ezmin.x;      // restart of the recurrence
            float gy = 0.f, gsum = 0.f;
            const float2* crow = cs + iy * g.nz;
            for (int iz = 0; iz < g.nz; ++iz) {
                const float2 c = crow[iz];
                ph = fmaf(c.x, pr, fmaf(c.y, pi, ph));
                if (FORCE) {
                    const float t = pr * c.y - pi * c.x;          // cos Im S - sin Re S (times w v)
                    gsum += t;
                    gy = fmaf((float)(iz - g.kz), t, gy);
                }
                const float nr = pr * ezstep.x - pi * ezstep.y;
                pi = pr * ezstep.y + pi * ezstep.x;
                pr = nr;
            }
            if (FORCE) {
                fx = fmaf((float)mx, gsum, fx);
                fy = fmaf((float)(iy - g.ky), gsum, fy);
                fz += gy;
            }
        }
    }
    // phi = (4 pi/V) sum; field per unit charge f = -(4 pi/V) sum k t  (F_i = q_i f_i; a-9 applies q_i)
    if (on) out[s] = make_float4(-g.four_pi_over_V * g.kfac[0] * fx, -g.four_pi_over_V * g.kfac[1] * fy,
                                 -g.four_pi_over_V * g.kfac[2] * fz, g.four_pi_over_V * ph);
}

// Reciprocal part into ctx->rec_out (same layout as the PME gather's output); E_rec into scal[1].
int ewald_recip_run(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3], double alpha,
                    const int kmax[3], bool want_force, cudaStream_t st)
{
    EwaldGeom g;
    g.kx = kmax[0]; g.ky = kmax[1]; g.kz = kmax[2];
    g.ny = 2 * g.ky + 1; g.nz = 2 * g.kz + 1;
    g.ntab = g.kx + 1 + g.ny + g.nz;
    g.nk = (g.kx + 1) * g.ny * g.nz;
    for (int d = 0; d < 3; ++d) { g.L[d] = box[d]; g.kfac[d] = (float)(2.0 * M_PI / box[d]); }
    g.four_pi_over_V = (float)(4.0 * M_PI / (box[0] * box[1] * box[2]));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->ew_tab, sizeof(float2) * (size_t)g.ntab * n));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->ew_sf, sizeof(float2) * (size_t)g.nk));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->rec_out, sizeof(float4) * n));
    float2* E = (float2*)ctx->ew_tab.p;
    float2* S = (float2*)ctx->ew_sf.p;
    {
        StageTimer tm(ctx, SQEQ_T_SPREAD, st);          // stage slots of the PME path: tables + S(k) ~ "spread"
        k_ewald_tables<<<dim3(ceil_div(n, 128), g.ntab), 128, 0, st>>>(n, pos, nl->perm, g, E);
        KERNEL_CHECK(ctx);
        const size_t sm = sizeof(float2) * (size_t)EW_CHUNK * (g.ntab + 1);
        CUDA_TRY(ctx, cudaFuncSetAttribute(k_ewald_sf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        k_ewald_sf<<<ceil_div(g.nk, 256), 256, sm, st>>>(n, E, (const float4*)ctx->xq.p, g, S);
        KERNEL_CHECK(ctx);
    }
    {
        StageTimer tm(ctx, SQEQ_T_INFLUENCE, st);
        double* e_out = (double*)ctx->scal.p + 1;
        CUDA_TRY(ctx, cudaMemsetAsync(e_out, 0, sizeof(double), st));
        k_ewald_coef<<<ceil_div(g.nk, 256), 256, 0, st>>>(g, alpha, S, e_out);
        KERNEL_CHECK(ctx);
    }
    {
        StageTimer tm(ctx, SQEQ_T_GATHER, st);
        const size_t sm = sizeof(float2) * (size_t)g.ny * g.nz;
        if (want_force) {
            CUDA_TRY(ctx, cudaFuncSetAttribute(k_ewald_gather<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            k_ewald_gather<true><<<ceil_div(n, 128), 128, sm, st>>>(n, E, S, g, (float4*)ctx->rec_out.p);
        } else {
            CUDA_TRY(ctx, cudaFuncSetAttribute(k_ewald_gather<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            k_ewald_gather<false><<<ceil_div(n, 128), 128, sm, st>>>(n, E, S, g, (float4*)ctx->rec_out.p);
        }
        KERNEL_CHECK(ctx);
    }
    return SQEQ_OK;
}

// OpenMM's tuning heuristics, which the paper says it uses: alpha = sqrt(-ln 2 delta)/rc; the
// smallest kmax_d with kmax sqrt(L_d alpha)/20 exp(-(pi kmax/(L_d alpha))^2) < delta (regular Ewald); grid_d =
// ceil(2 alpha L_d/(3 delta^(1/5))) rounded up to an even number with factors 2, 3, 5 only (PME).  The formulas are
// recalled from OpenMM's documentation, not printed in the paper (reading G17).
extern "C" int sqeq_ewald_params(const double box[3], double rc, double delta, double* alpha, int kmax[3], int grid[3])
{
    if (!box || !(rc > 0.0) || !(delta > 0.0) || !(delta < 0.5)) return SQEQ_EINVAL;
    const double a = sqrt(-log(2.0 * delta)) / rc;
    if (alpha) *alpha = a;
    for (int d = 0; d < 3; ++d) {
        if (!(box[d] > 0.0)) return SQEQ_EINVAL;
        if (kmax) {
            int k = 1;
            while (k < 4096 && k * sqrt(box[d] * a) / 20.0 * exp(-pow(M_PI * k / (box[d] * a), 2.0)) >= delta) ++k;
            kmax[d] = k;
        }
        if (grid) {
            int K = (int)ceil(2.0 * a * box[d] / (3.0 * pow(delta, 0.2)));
            if (K < 8) K = 8;
            for (;; ++K) {
                if (K & 1) continue;
                int r = K;
                for (int p : {2, 3, 5}) while (r % p == 0) r /= p;
                if (r == 1) break;
            }
            grid[d] = K;
        }
    }
    return SQEQ_OK;
}

extern "C" int sqeq_coulomb_ewald(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const float* q,
                                  const double box[3], double rc, double alpha, const int kmax[3], float* phi,
                                  float* force, double* energy)
{
    if (!ctx) return SQEQ_EINVAL;
    const int grid_dummy[3] = {8, 8, 8};
    SQEQ_TRY(validate_coulomb_args(ctx, nl, n, box, rc, alpha, grid_dummy, 6, "sqeq_coulomb_ewald"));
    if (!pos || !q || !kmax) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_ewald: NULL argument");
    for (int d = 0; d < 3; ++d)
        if (kmax[d] < 1 || kmax[d] > 128)
            return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_ewald: kmax[%d] = %d must be in [1, 128]", d, kmax[d]);
    if ((size_t)(2 * kmax[1] + 1) * (2 * kmax[2] + 1) * sizeof(float2) > 200 * 1024)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_ewald: (2 kmax_y + 1)(2 kmax_z + 1) coefficients do not fit shared memory; "
                                           "use PME for systems this large");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const bool want_force = force != nullptr;
    SQEQ_TRY(prep_atoms(ctx, nl, pos, q, nullptr, st));
    SQEQ_TRY(ewald_recip_run(ctx, nl, n, pos, box, alpha, kmax, want_force, st));
    ctx->overlap_now = false;
    SQEQ_TRY(realspace_run(ctx, nl, rc, alpha, want_force, st));
    SQEQ_TRY(assemble_run(ctx, nl, alpha, phi, force, energy != nullptr, false, st));
    ctx->last_had_force = want_force;
    ctx->last_n = n;
    ctx->energy_pending = energy != nullptr;
    if (energy) SQEQ_TRY(sqeq_energy_fetch(ctx, energy));
    return SQEQ_OK;
}
