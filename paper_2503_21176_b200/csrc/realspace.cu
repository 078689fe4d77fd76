// realspace.cu -- per-evaluation atom re-gather (prep) and the erfc-screened real-space pair sum,
// Eq. 3 restricted to r < rc over the neighbour list (step a-3), plus the final
// assembly with the self term of Eq. 5 (step a-9).
//
// One warp per atom row: lanes stride over the row's packed entries (coalesced 128 B list loads),
// gather the neighbour's float4 (x,y,z,q) from the cell-major array (L1/L2 resident), apply the
// image shift from a 27-entry shared table, accumulate phi and F in registers, then a shuffle
// reduction -- no atomics (the paper's ELLPACK row sum, without the padding).
#include <math.h>
#include <stdlib.h>

#include "common.cuh"

struct PrepGeom {
    double L[3];
    int    K[3];   // 0 => no PME coordinates wanted
};

__global__ void k_prep(int64_t n, const float* __restrict__ pos, const float* __restrict__ q,
                       const int* __restrict__ perm, const char4* __restrict__ wrapc, PrepGeom g,
                       float4* __restrict__ xq, float4* __restrict__ frac, int4* __restrict__ base)
{
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int o = perm[s];
    const char4 w = wrapc[s];
    const int wd[3] = {w.x, w.y, w.z};
    const float qi = q ? q[o] : 0.f;
    float xw[3], fw[3];
    int f[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        // same periodic image as at build time, so the list's image codes stay valid
        double x = (double)pos[3 * (int64_t)o + d] - (double)wd[d] * g.L[d];
        xw[d] = (float)x;
        if (g.K[0] > 0) {
            // fractional grid coordinate in fp64 (an fp32 product x*K/L loses ~1e-5 of a cell at x~150)
            double u = x / g.L[d];
            u -= floor(u);
            u *= (double)g.K[d];
            int fi = (int)u;
            if (fi >= g.K[d]) { fi -= g.K[d]; u -= (double)g.K[d]; }
            double wv = u - (double)fi;
            fw[d] = wv < 0.0 ? 0.f : (float)wv;
            f[d] = fi;
        }
    }
    xq[s] = make_float4(xw[0], xw[1], xw[2], qi);
    if (g.K[0] > 0) {
        frac[s] = make_float4(fw[0], fw[1], fw[2], qi);
        base[s] = make_int4(f[0], f[1], f[2], 0);
    }
}

__global__ void k_prep_charges(int64_t n, const float* __restrict__ qf, const double* __restrict__ qd,
                               const int* __restrict__ perm, float4* __restrict__ xq,
                               float4* __restrict__ frac)
{
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int o = perm[s];
    const float qi = qf ? qf[o] : (float)qd[o];
    xq[s].w = qi;
    frac[s].w = qi;
}

int prep_atoms(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* pos, const float* q, const int* K,
               cudaStream_t st)
{
    const int64_t n = nl->n;
    SQEQ_TRY(sqeq_reserve(ctx, ctx->xq, sizeof(float4) * (n + 32)));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->frac, sizeof(float4) * n));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->base, sizeof(int4) * n));
    PrepGeom g;
    for (int d = 0; d < 3; ++d) { g.L[d] = nl->box[d]; g.K[d] = K ? K[d] : 0; }
    ctx->gc.valid = false;                      // new positions: the geometry cache is stale
    ctx->geom_serial++;
    StageTimer tm(ctx, SQEQ_T_PREP, st);
    k_prep<<<ceil_div(n, 256), 256, 0, st>>>(n, pos, q, nl->perm, nl->wrapc, g, (float4*)ctx->xq.p,
                                              (float4*)ctx->frac.p, (int4*)ctx->base.p);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

int prep_charges(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* q_f, const double* q_d,
                 cudaStream_t st)
{
    const int64_t n = nl->n;
    StageTimer tm(ctx, SQEQ_T_PREP, st);
    k_prep_charges<<<ceil_div(n, 256), 256, 0, st>>>(n, q_f, q_d, nl->perm, (float4*)ctx->xq.p,
                                                      (float4*)ctx->frac.p);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

// ------------------------------------------------------------------------------------------------
struct RealParams {
    float Lx, Ly, Lz;
    float rc2;
    float pa;        // ERFC_P alpha (erfc_from_exp)
    float c2;        // 2 alpha / sqrt(pi)
    float na2l2e;    // -alpha^2 log2(e):  exp(-alpha^2 r^2) = 2^(na2l2e r^2)
};

// MUFU wrappers (one XU instruction each, <= 2 ulp; flush-to-zero is harmless here)
__device__ __forceinline__ float mufu_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x)   { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x)   { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// erfc(x) = exp(-x^2) t P5(t), t = 1/(1 + 0.4 x), x >= 0, given ex = exp(-x^2).
// The form is Abramowitz & Stegun 7.1.26 with one more term and its own constant in t; the coefficients
// are a weighted minimax (Lawson) fit of erfcx(x) = exp(x^2) erfc(x) made for this library: max |error|
// of erfc 2.8e-8 in exact arithmetic, 3.6e-8 rms / 4.2e-7 max once evaluated in fp32 (the fp32 rounding
// of the product dominates) -- 1 MUFU.RCP + 7 FP32 ops instead of the ~40-instruction erfcf, and it
// shares the exp(-alpha^2 r^2) the force needs anyway.
// Called with r and pa = 0.4 alpha, so that the product alpha r is never formed on its own.
#define ERFC_P 0.4
__device__ __forceinline__ float erfc_from_exp(float r, float pa, float ex)
{
    const float t = mufu_rcp(fmaf(pa, r, 1.f));
    float p = -0.20025848511103075f;
    p = fmaf(p, t, 0.7091442915149763f);
    p = fmaf(p, t, -0.370903111156111f);
    p = fmaf(p, t, 0.468270358550566f);
    p = fmaf(p, t, 0.16182505660344682f);
    p = fmaf(p, t, 0.23192186199974116f);
    return p * t * ex;
}

template <bool FORCE>
__global__ void __launch_bounds__(256)
k_real(int64_t n, const float4* __restrict__ xq, const int64_t* __restrict__ row_start,
       const int* __restrict__ row_len, const uint32_t* __restrict__ nbr, RealParams p,
       float4* __restrict__ out)
{
    __shared__ float4 sh[32];
    if (threadIdx.x < 32) {
        int img = threadIdx.x < 27 ? threadIdx.x : 13;
        sh[threadIdx.x] = make_float4((img / 9 - 1) * p.Lx, ((img / 3) % 3 - 1) * p.Ly, (img % 3 - 1) * p.Lz, 0.f);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int64_t s = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (s >= n) return;
    const float4 xi = xq[s];
    const uint32_t* __restrict__ row = nbr + row_start[s];
    const int len = row_len[s];
    float phi = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
    // branch-free body: a lane outside rc contributes q_j * 0, so the two unrolled iterations interleave
#pragma unroll 2
    for (int k = lane; k < len; k += 32) {
        const uint32_t e = __ldg(row + k);
        const float4 xj = __ldg(xq + (e & 0x07ffffffu));
        const float4 s4 = sh[e >> 27];
        // d = r_i - (r_j + shift)
        const float dx = (xi.x - xj.x) - s4.x;
        const float dy = (xi.y - xj.y) - s4.y;
        const float dz = (xi.z - xj.z) - s4.z;
        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        const float qj = r2 < p.rc2 ? xj.w : 0.f;
        const float rinv = mufu_rsqrt(r2);
        const float ex = mufu_ex2(p.na2l2e * r2);             // exp(-alpha^2 r^2)
        const float t = erfc_from_exp(r2 * rinv, p.pa, ex) * rinv;   // erfc(alpha r)/r
        phi = fmaf(qj, t, phi);
        if (FORCE) {
            const float gq = qj * fmaf(p.c2, ex, t) * (rinv * rinv);
            fx = fmaf(gq, dx, fx);
            fy = fmaf(gq, dy, fy);
            fz = fmaf(gq, dz, fz);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        phi += __shfl_xor_sync(0xffffffffu, phi, o);
        if (FORCE) {
            fx += __shfl_xor_sync(0xffffffffu, fx, o);
            fy += __shfl_xor_sync(0xffffffffu, fy, o);
            fz += __shfl_xor_sync(0xffffffffu, fz, o);
        }
    }
    // the field sum_j q_j g d (no q_i factor: a-9 applies it, or not in field mode)
    if (lane == 0) out[s] = make_float4(fx, fy, fz, phi);
}

// The same sum with the neighbourhood STAGED IN SHARED MEMORY (list format 1, cellgroup.cuh): one block
// per group of 2x2x2 cells.  The block copies the group's neighbourhood -- every piece a contiguous run
// of the cell-major float4 array, coalesced -- into shared memory with the piece's image shift already
// added, then each warp takes rows of the group's own atoms: 16-bit local indices from the list (64 B
// per warp load), neighbour (x,y,z,q) by LDS.128 instead of a scattered global gather, no per-pair
// shift, same arithmetic as k_real.
#ifndef REAL_NT
#define REAL_NT 512
#endif
#ifndef REAL_BATCH_F
#define REAL_BATCH_F 8      // entry loads in flight, force kernel
#endif
#ifndef REAL_BATCH_P
#define REAL_BATCH_P 16     // entry loads in flight, potential-only kernel
#endif
#ifndef REAL_BPS_F
#define REAL_BPS_F 3        // blocks per SM the register budget is set for, force kernel
#endif
#ifndef REAL_BPS_P
#define REAL_BPS_P 4        // ... potential-only kernel
#endif
#ifndef REAL_BPS_C
#define REAL_BPS_C 3        // ... cache-writing variants
#endif
#ifndef REAL_BATCH_C
#define REAL_BATCH_C 4      // entry loads in flight, cache-writing variants
#endif
__device__ __forceinline__ float4 lds128(unsigned addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// SCALED: the list entries are byte offsets into the staged array (local index * 16, nl->lshift = 4)
// LEAN: 32 registers (four blocks per SM would fit) and 4 loads in flight -- the variant launched as a
// PERSISTENT grid of a few blocks per SM beside the PME kernels (SQEQ_OVERLAP=1), each block walking over
// cell groups, so that the register file and shared memory have room for both.
// CACHE (geometry cache): also write, per row, the COMPACT list of the entries with
// r < rc (same 16-bit entry, same row offset) and their t = erfc(alpha r)/r.  Later evaluations on the same
// geometry (Krylov iterations, the second force evaluation of an MD step) use that list: potentials are a sparse
// product over t (k_real_cached: no MUFU, no skin entries), forces run this kernel over the compact rows.
struct RealCache {
    uint16_t* idx;     // [n_slots] compact rows, padded to whole warps with the dummy entry
    float*    t;       // [n_slots]
    int*      len;     // [n] entries of the compact row
};

template <bool FORCE, bool SCALED, bool LEAN = false, int CACHE = 0>
__global__ void __launch_bounds__(REAL_NT, CACHE ? REAL_BPS_C : (LEAN ? 4 : (FORCE ? REAL_BPS_F : REAL_BPS_P)))
k_real_staged(const float4* __restrict__ xq, const int* __restrict__ cell_start, GroupGeom gg,
              const int64_t* __restrict__ row_start, const int* __restrict__ row_len,
              const uint16_t* __restrict__ nbr, const longlong2* __restrict__ grp_slice, RealParams p,
              int ngroups, float4* __restrict__ out, RealCache rcache)
{
    extern __shared__ __align__(16) float4 xs[];               // [neighbourhood population + 1]
    __shared__ GroupPiece pieces[GRP_MAXPIECE];
    __shared__ int s_scratch, s_roff[GRP_G * GRP_G], s_rpre[GRP_G * GRP_G + 1];
    for (int grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
    if (grp != (int)blockIdx.x) __syncthreads();               // the previous group's shared state is still being read
    if (grp_slice) {
        // the group's rows sit in one contiguous slice of the list (k_pairs reserves it per group): ask for it
        // in L2 now, so that the entry loads below meet L2 latency instead of DRAM latency (not for the compact
        // rows of the geometry cache, which fill only a part of each row's slots)
        const longlong2 sl = grp_slice[grp];
        const char* base = (const char*)(nbr + sl.x);
        const long long bytes = sl.y * (long long)sizeof(uint16_t);
        for (long long o = (long long)threadIdx.x * 128; o < bytes; o += (long long)REAL_NT * 128)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(base + o));
    }
    const GroupInfo gi = group_layout(gg, cell_start, grp, pieces, &s_scratch);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int r = 0; r < GRP_G * GRP_G; ++r) {
            s_rpre[r] = acc;
            const int ix = r / GRP_G, iy = r % GRP_G;
            if (ix < gi.ge[0] && iy < gi.ge[1]) {
                const int colw = ((gi.c0[0] + ix) * gg.nc[1] + gi.c0[1] + iy) * gg.nc[2] + gi.c0[2];
                const int beg = cell_start[colw];
                s_roff[r] = beg - acc;                         // sorted index = own-atom number + s_roff[range]
                acc += cell_start[colw + gi.ge[2]] - beg;
            } else {
                s_roff[r] = 0;
            }
        }
        s_rpre[GRP_G * GRP_G] = acc;
        // the dummy slot the padding entries of the rows point to: outside every cutoff, charge 0
        xs[gi.pop] = make_float4(1e15f, 1e15f, 1e15f, 0.f);
    }
    // stage: one warp per piece at a time
    const int np = gi.ncol * 3;
    for (int ip = wid; ip < np; ip += REAL_NT / 32) {
        const GroupPiece pc = pieces[ip];
        if (pc.len == 0) continue;
        const float sx = (pc.code / 9 - 1) * p.Lx, sy = ((pc.code / 3) % 3 - 1) * p.Ly, sz = (pc.code % 3 - 1) * p.Lz;
        for (int k = lane; k < pc.len; k += 32) {
            float4 v = __ldg(xq + pc.gbeg + k);
            v.x += sx; v.y += sy; v.z += sz;
            xs[pc.lbase + k] = v;
        }
    }
    __syncthreads();
    const int natoms = s_rpre[GRP_G * GRP_G];
    const int p1 = s_rpre[1], p2 = s_rpre[2], p3 = s_rpre[3];
    static_assert(GRP_G * GRP_G == 4, "range lookup below is written for four ranges");
    for (int ia = wid; ia < natoms; ia += REAL_NT / 32) {
        const int s = ia + s_roff[(ia >= p1) + (ia >= p2) + (ia >= p3)];
        const float4 xi = __ldg(xq + s);
        // rows are padded to whole 32-entry steps (the padding points at the dummy slot), so the loop is
        // uniform over the warp
        const int64_t r0 = row_start[s];
        const uint16_t* __restrict__ row = nbr + r0 + lane;
        const int nst = (row_len[s] + 31) >> 5;
        const unsigned xs_addr = (unsigned)__cvta_generic_to_shared(xs);
        float phi = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
        unsigned ccnt = 0;                                         // CACHE: entries of the compact row so far
        const unsigned lt = (1u << lane) - 1u;
        uint16_t* __restrict__ crow_i = CACHE ? rcache.idx + r0 : nullptr;
        float* __restrict__ crow_t = CACHE ? rcache.t + r0 : nullptr;
        auto pair = [&](unsigned e) {
            const float4 xj = SCALED ? lds128(xs_addr + e) : xs[e];
            const float dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const bool inr = r2 < p.rc2;
            const float qj = inr ? xj.w : 0.f;
            const float rinv = mufu_rsqrt(r2);
            const float ex = mufu_ex2(p.na2l2e * r2);             // exp(-alpha^2 r^2)
            const float t = erfc_from_exp(r2 * rinv, p.pa, ex) * rinv;   // erfc(alpha r)/r
            phi = fmaf(qj, t, phi);
            if (FORCE) {
                const float gq = qj * fmaf(p.c2, ex, t) * (rinv * rinv);
                fx = fmaf(gq, dx, fx);
                fy = fmaf(gq, dy, fy);
                fz = fmaf(gq, dz, fz);
            }
            if (CACHE) {
                const unsigned m = __ballot_sync(0xffffffffu, inr);
                if (inr) {
                    const unsigned d = ccnt + __popc(m & lt);
                    crow_i[d] = (uint16_t)e;
                    crow_t[d] = t;
                }
                ccnt += __popc(m);
            }
        };
        // four entry loads in flight ahead of the four pair evaluations that use them
        // the entry loads of B steps are issued together ahead of the B pair evaluations that use them
        // (B = 16/8/4 while the row lasts): the potential-only kernel has registers for 16 in flight, the
        // force kernel for 4
        constexpr int BMAX = CACHE ? REAL_BATCH_C : (LEAN ? 4 : (FORCE ? REAL_BATCH_F : REAL_BATCH_P));
        int it = 0;
        if (BMAX >= 16)
            for (; it + 16 <= nst; it += 16) {
                unsigned e[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) e[k] = __ldg(row + 32 * (it + k));
#pragma unroll
                for (int k = 0; k < 16; ++k) pair(e[k]);
            }
        if (BMAX >= 8)
            for (; it + 8 <= nst; it += 8) {
                unsigned e[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) e[k] = __ldg(row + 32 * (it + k));
#pragma unroll
                for (int k = 0; k < 8; ++k) pair(e[k]);
            }
        for (; it + 4 <= nst; it += 4) {
            const unsigned e0 = __ldg(row + 32 * it), e1 = __ldg(row + 32 * it + 32), e2 = __ldg(row + 32 * it + 64),
                           e3 = __ldg(row + 32 * it + 96);
            pair(e0); pair(e1); pair(e2); pair(e3);
        }
        if (it + 2 <= nst) {
            const unsigned e0 = __ldg(row + 32 * it), e1 = __ldg(row + 32 * it + 32);
            pair(e0); pair(e1);
            it += 2;
        }
        if (it < nst) pair(__ldg(row + 32 * it));
        if (CACHE) {
            // pad the compact row to whole warps with the dummy entry (charge 0, t = g = 0)
            const unsigned padn = (ccnt + 31u) & ~31u;
            if (ccnt + lane < padn) {
                crow_i[ccnt + lane] = (uint16_t)(SCALED ? gi.pop << 4 : gi.pop);
                crow_t[ccnt + lane] = 0.f;
            }
            if (lane == 0) rcache.len[s] = (int)ccnt;
        }
        if (FORCE) {
            const float v = warp_reduce4(fx, fy, fz, phi, lane);        // lanes 0 / 8 / 16 / 24: fx / fy / fz / phi
            if ((lane & 7) == 0) ((float*)(out + s))[lane >> 3] = v;
        } else {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) phi += __shfl_xor_sync(0xffffffffu, phi, o);
            if (lane == 0) out[s] = make_float4(0.f, 0.f, 0.f, phi);
        }
    }
    }   // groups
}

// The same sums over the geometry cache a CACHE pass of k_real_staged left behind (NEXT-1): per row the compact
// list of in-range entries with t = erfc(alpha r)/r (MODE 0: potential, phi_i = sum_j q_j t_ij -- a sparse
// matrix-vector product, 6 B per entry, no MUFU, the block stages only the neighbourhood's CHARGES) or
// g (MODE 1: per-unit-charge field, f_i = sum_j q_j g_ij (r_i - r_j), staged float4 as above).  HBM-bound: the
// loads of 8 steps are issued ahead of their use.
template <int MODE, bool SCALED>
__global__ void __launch_bounds__(REAL_NT, MODE == 2 ? 2 : 3)
k_real_cached(const float4* __restrict__ xq, const int* __restrict__ cell_start, GroupGeom gg,
              const int64_t* __restrict__ row_start, RealParams p, int ngroups, float4* __restrict__ out,
              RealCache rcache)
{
    extern __shared__ __align__(16) float4 xs[];               // MODE 1: float4 [pop + 1]; MODE 0: float [pop + 1]
    __shared__ GroupPiece pieces[GRP_MAXPIECE];
    __shared__ int s_scratch, s_roff[GRP_G * GRP_G], s_rpre[GRP_G * GRP_G + 1];
    float* qs = (float*)xs;
    const int grp = blockIdx.x;
    const GroupInfo gi = group_layout(gg, cell_start, grp, pieces, &s_scratch);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int r = 0; r < GRP_G * GRP_G; ++r) {
            s_rpre[r] = acc;
            const int ix = r / GRP_G, iy = r % GRP_G;
            if (ix < gi.ge[0] && iy < gi.ge[1]) {
                const int colw = ((gi.c0[0] + ix) * gg.nc[1] + gi.c0[1] + iy) * gg.nc[2] + gi.c0[2];
                const int beg = cell_start[colw];
                s_roff[r] = beg - acc;
                acc += cell_start[colw + gi.ge[2]] - beg;
            } else {
                s_roff[r] = 0;
            }
        }
        s_rpre[GRP_G * GRP_G] = acc;
        if (MODE == 0) qs[gi.pop] = 0.f; else xs[gi.pop] = make_float4(1e15f, 1e15f, 1e15f, 0.f);
    }
    const int np = gi.ncol * 3;
    for (int ip = wid; ip < np; ip += REAL_NT / 32) {
        const GroupPiece pc = pieces[ip];
        if (pc.len == 0) continue;
        if (MODE == 0) {
            for (int k = lane; k < pc.len; k += 32) qs[pc.lbase + k] = __ldg(&xq[pc.gbeg + k].w);
        } else {
            const float sx = (pc.code / 9 - 1) * p.Lx, sy = ((pc.code / 3) % 3 - 1) * p.Ly, sz = (pc.code % 3 - 1) * p.Lz;
            for (int k = lane; k < pc.len; k += 32) {
                float4 v = __ldg(xq + pc.gbeg + k);
                v.x += sx; v.y += sy; v.z += sz;
                xs[pc.lbase + k] = v;
            }
        }
    }
    __syncthreads();
    const int natoms = s_rpre[GRP_G * GRP_G];
    const int p1 = s_rpre[1], p2 = s_rpre[2], p3 = s_rpre[3];
    const unsigned xs_addr = (unsigned)__cvta_generic_to_shared(xs);
    static_assert(MODE == 0, "only the potential is taken from the cache; forces run k_real_staged over the compact rows");
    const float* __restrict__ cval = rcache.t;
    constexpr int NW = REAL_NT / 32;
    for (int base = 0; base < natoms; base += NW * 32) {
    // lane l fetches the row offset and length of the l-th row this warp will take: one round trip for all of
    // them instead of one per row
    int my_s = 0, my_len = 0;
    int64_t my_r0 = 0;
    {
        const int ia = base + wid + NW * lane;
        if (ia < natoms) {
            my_s = ia + s_roff[(ia >= p1) + (ia >= p2) + (ia >= p3)];
            my_r0 = row_start[my_s];
            my_len = rcache.len[my_s];
        }
    }
    for (int l = 0; l < 32; ++l) {
        const int ia = base + wid + NW * l;
        if (ia >= natoms) break;
        const int s = __shfl_sync(0xffffffffu, my_s, l);
        const int len_s = __shfl_sync(0xffffffffu, my_len, l);
        // A lane takes FOUR consecutive entries of every 128-entry chunk of the row: one 8-byte load of the
        // entries and one 16-byte load of their values per lane and chunk (rows start on multiples of 32
        // entries, so both are aligned; a quad is either wholly inside the padded row or wholly outside).  The
        // loads of up to four chunks -- a whole typical row of ~300 in-range entries -- are issued before the
        // first use: the kernel is a stream from HBM.
        const int64_t r0 = __shfl_sync(0xffffffffu, my_r0, l) + 4 * lane;
        const uint2* __restrict__ ri = (const uint2*)(rcache.idx + r0);
        const float4* __restrict__ rv = (const float4*)(cval + r0);
        const float4* __restrict__ rt = (const float4*)(rcache.t + r0);
        const int padlen = (len_s + 31) & ~31;
        float4 xi = make_float4(0.f, 0.f, 0.f, 0.f);
        if (MODE != 0) xi = __ldg(xq + s);
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
        auto term = [&](unsigned e, float v, float vt) {          // e: 16-bit entry in the low half
            if (MODE == 0) {
                float qj;
                const unsigned a = xs_addr + (SCALED ? e >> 2 : e << 2);
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(qj) : "r"(a));
                a3 = fmaf(qj, v, a3);
            } else {
                const float4 xj = SCALED ? lds128(xs_addr + e) : xs[e];
                const float gq = xj.w * v;
                a0 = fmaf(gq, xi.x - xj.x, a0);
                a1 = fmaf(gq, xi.y - xj.y, a1);
                a2 = fmaf(gq, xi.z - xj.z, a2);
                if (MODE == 2) a3 = fmaf(xj.w, vt, a3);
            }
        };
        constexpr int B = MODE == 2 ? 2 : 4;                       // chunks in flight
        for (int c0 = 0; c0 < padlen; c0 += 128 * B) {
            uint2 e[B];
            float4 v[B], vt[B];
#pragma unroll
            for (int k = 0; k < B; ++k) {
                const bool on = c0 + 128 * k + 4 * lane < padlen;
                e[k] = make_uint2(0u, 0u);                          // entry 0 with value 0: contributes nothing
                v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                vt[k] = v[k];
                if (on) {
                    e[k] = __ldg(ri + ((c0 + 128 * k) >> 2));
                    v[k] = __ldg(rv + ((c0 + 128 * k) >> 2));
                    if (MODE == 2) vt[k] = __ldg(rt + ((c0 + 128 * k) >> 2));
                }
            }
#pragma unroll
            for (int k = 0; k < B; ++k) {
                if (c0 + 128 * k < padlen) {                        // uniform over the warp
                    term(e[k].x & 0xffffu, v[k].x, vt[k].x);
                    term(e[k].x >> 16, v[k].y, vt[k].y);
                    term(e[k].y & 0xffffu, v[k].z, vt[k].z);
                    term(e[k].y >> 16, v[k].w, vt[k].w);
                }
            }
        }
        if (MODE == 0) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) a3 += __shfl_xor_sync(0xffffffffu, a3, o);
            if (lane == 0) out[s] = make_float4(0.f, 0.f, 0.f, a3);
        } else {
            const float v = warp_reduce4(a0, a1, a2, a3, lane);
            if ((lane & 7) == 0) ((float*)(out + s))[lane >> 3] = v;
        }
    }
    }   // row batches
}

// NEXT-1, batched right-hand sides: the same sparse product for NV charge vectors in ONE pass over the cache
// (phi^v_i = sum_j t_ij q^v_j, v < NV).  The cache stream (6 B per entry) is what bounds k_real_cached; here it is read
// once for all vectors.  The neighbourhood's charges are staged interleaved (NV floats per slot: one LDS.64 / LDS.128 per
// entry), qs_sorted = the vectors in the list's sorted order [NV][n], out = [NV][n] in sorted order.
template <int NV, bool SCALED>
__global__ void __launch_bounds__(REAL_NT, 3)
k_real_cached_multi(const float* __restrict__ qs_sorted, int64_t n, const int* __restrict__ cell_start, GroupGeom gg,
                    const int64_t* __restrict__ row_start, int ngroups, float* __restrict__ out, RealCache rcache)
{
    static_assert(NV == 2 || NV == 4, "two or four vectors per pass");
    extern __shared__ __align__(16) float4 xs[];               // float [pop + 1][NV]
    __shared__ GroupPiece pieces[GRP_MAXPIECE];
    __shared__ int s_scratch, s_roff[GRP_G * GRP_G], s_rpre[GRP_G * GRP_G + 1];
    float* qs = (float*)xs;
    const int grp = blockIdx.x;
    const GroupInfo gi = group_layout(gg, cell_start, grp, pieces, &s_scratch);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int r = 0; r < GRP_G * GRP_G; ++r) {
            s_rpre[r] = acc;
            const int ix = r / GRP_G, iy = r % GRP_G;
            if (ix < gi.ge[0] && iy < gi.ge[1]) {
                const int colw = ((gi.c0[0] + ix) * gg.nc[1] + gi.c0[1] + iy) * gg.nc[2] + gi.c0[2];
                const int beg = cell_start[colw];
                s_roff[r] = beg - acc;
                acc += cell_start[colw + gi.ge[2]] - beg;
            } else {
                s_roff[r] = 0;
            }
        }
        s_rpre[GRP_G * GRP_G] = acc;
        for (int v = 0; v < NV; ++v) qs[gi.pop * NV + v] = 0.f;    // the slot the row padding points at
    }
    const int np = gi.ncol * 3;
    for (int ip = wid; ip < np; ip += REAL_NT / 32) {
        const GroupPiece pc = pieces[ip];
        for (int k = lane; k < pc.len; k += 32)
#pragma unroll
            for (int v = 0; v < NV; ++v) qs[(pc.lbase + k) * NV + v] = __ldg(qs_sorted + (int64_t)v * n + pc.gbeg + k);
    }
    __syncthreads();
    const int natoms = s_rpre[GRP_G * GRP_G];
    const int p1 = s_rpre[1], p2 = s_rpre[2], p3 = s_rpre[3];
    const unsigned xs_addr = (unsigned)__cvta_generic_to_shared(xs);
    constexpr int NW = REAL_NT / 32;
    for (int base = 0; base < natoms; base += NW * 32) {
        int my_s = 0, my_len = 0;
        int64_t my_r0 = 0;
        {
            const int ia = base + wid + NW * lane;
            if (ia < natoms) {
                my_s = ia + s_roff[(ia >= p1) + (ia >= p2) + (ia >= p3)];
                my_r0 = row_start[my_s];
                my_len = rcache.len[my_s];
            }
        }
        for (int l = 0; l < 32; ++l) {
            const int ia = base + wid + NW * l;
            if (ia >= natoms) break;
            const int s = __shfl_sync(0xffffffffu, my_s, l);
            const int len_s = __shfl_sync(0xffffffffu, my_len, l);
            const int64_t r0 = __shfl_sync(0xffffffffu, my_r0, l) + 4 * lane;
            const uint2* __restrict__ ri = (const uint2*)(rcache.idx + r0);
            const float4* __restrict__ rv = (const float4*)(rcache.t + r0);
            const int padlen = (len_s + 31) & ~31;
            float acc[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) acc[v] = 0.f;
            auto term = [&](unsigned e, float t) {                 // e: 16-bit entry (slot, or slot << 4 when SCALED)
                if (NV == 2) {
                    float q0, q1;
                    const unsigned a = xs_addr + (SCALED ? e >> 1 : e << 3);
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(q0), "=f"(q1) : "r"(a));
                    acc[0] = fmaf(q0, t, acc[0]);
                    acc[1] = fmaf(q1, t, acc[1]);
                } else {
                    const float4 qv = lds128(xs_addr + (SCALED ? e : e << 4));
                    acc[0] = fmaf(qv.x, t, acc[0]);
                    acc[1] = fmaf(qv.y, t, acc[1]);
                    acc[NV - 2] = fmaf(qv.z, t, acc[NV - 2]);
                    acc[NV - 1] = fmaf(qv.w, t, acc[NV - 1]);
                }
            };
            constexpr int B = 4;                                   // chunks of 128 entries in flight
            for (int c0 = 0; c0 < padlen; c0 += 128 * B) {
                uint2 e[B];
                float4 t[B];
#pragma unroll
                for (int k = 0; k < B; ++k) {
                    e[k] = make_uint2(0u, 0u);
                    t[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (c0 + 128 * k + 4 * lane < padlen) {
                        e[k] = __ldg(ri + ((c0 + 128 * k) >> 2));
                        t[k] = __ldg(rv + ((c0 + 128 * k) >> 2));
                    }
                }
#pragma unroll
                for (int k = 0; k < B; ++k) {
                    if (c0 + 128 * k < padlen) {
                        term(e[k].x & 0xffffu, t[k].x);
                        term(e[k].x >> 16, t[k].y);
                        term(e[k].y & 0xffffu, t[k].z);
                        term(e[k].y >> 16, t[k].w);
                    }
                }
            }
#pragma unroll
            for (int v = 0; v < NV; ++v) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) acc[v] += __shfl_xor_sync(0xffffffffu, acc[v], o);
            }
            if (lane < NV) {
                float r = acc[0];
#pragma unroll
                for (int v = 1; v < NV; ++v) r = lane == v ? acc[v] : r;
                out[(int64_t)lane * n + s] = r;
            }
        }
    }
}

// The same sparse product with the rows STREAMED BY THE BULK-COPY ENGINE (TMA 1-D, cp.async.bulk + mbarrier): one
// lane of a warp asks for a whole row -- its compact entries and their t, two contiguous 16-byte-aligned stretches of
// the cache -- to be copied into the warp's shared-memory buffer, and the copy of the NEXT row is in flight while the
// warp sums the current one (two buffers and two mbarriers per warp).  The lanes then read entries and values from
// shared memory with conflict-free vector loads: no per-lane global loads, predicates or address arithmetic, and the
// bytes in flight do not depend on registers.  Rows longer than the buffer (RCAP entries) take the kernel above.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned phase)
{
    unsigned ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(bar), "r"(phase) : "memory");
    } while (!ok);
}

template <bool SCALED, int RCAP>
__global__ void __launch_bounds__(REAL_NT, 2)
k_real_cached_tma(const float4* __restrict__ xq, const int* __restrict__ cell_start, GroupGeom gg,
                  const int64_t* __restrict__ row_start, RealParams p, int ngroups, float4* __restrict__ out,
                  RealCache rcache)
{
    constexpr int NW = REAL_NT / 32;
    constexpr int BUFB = RCAP * 6;                              // t [RCAP] fp32, then entries [RCAP] u16
    extern __shared__ __align__(128) unsigned char smem_tma[];  // NW x 2 buffers | charges [pop + 1]
    __shared__ __align__(8) unsigned long long bars[NW][2];
    __shared__ GroupPiece pieces[GRP_MAXPIECE];
    __shared__ int s_scratch, s_roff[GRP_G * GRP_G], s_rpre[GRP_G * GRP_G + 1];
    float* qs = (float*)(smem_tma + (size_t)NW * 2 * BUFB);
    const int grp = blockIdx.x;
    const GroupInfo gi = group_layout(gg, cell_start, grp, pieces, &s_scratch);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int r = 0; r < GRP_G * GRP_G; ++r) {
            s_rpre[r] = acc;
            const int ix = r / GRP_G, iy = r % GRP_G;
            if (ix < gi.ge[0] && iy < gi.ge[1]) {
                const int colw = ((gi.c0[0] + ix) * gg.nc[1] + gi.c0[1] + iy) * gg.nc[2] + gi.c0[2];
                const int beg = cell_start[colw];
                s_roff[r] = beg - acc;
                acc += cell_start[colw + gi.ge[2]] - beg;
            } else {
                s_roff[r] = 0;
            }
        }
        s_rpre[GRP_G * GRP_G] = acc;
        qs[gi.pop] = 0.f;
    }
    if (lane == 0) {
        mbar_init(smem_u32(&bars[wid][0]), 1);
        mbar_init(smem_u32(&bars[wid][1]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int np = gi.ncol * 3;
    for (int ip = wid; ip < np; ip += NW) {
        const GroupPiece pc = pieces[ip];
        for (int k = lane; k < pc.len; k += 32) qs[pc.lbase + k] = __ldg(&xq[pc.gbeg + k].w);
    }
    __syncthreads();
    const int natoms = s_rpre[GRP_G * GRP_G];
    const int p1 = s_rpre[1], p2 = s_rpre[2], p3 = s_rpre[3];
    const unsigned qs_addr = smem_u32(qs);
    unsigned char* mybuf = smem_tma + (size_t)wid * 2 * BUFB;
    unsigned phase0 = 0, phase1 = 0;
    for (int base = 0; base < natoms; base += NW * 32) {
        // lane l holds the row offset and length of the l-th row this warp will take
        int my_s = 0, my_len = 0;
        int64_t my_r0 = 0;
        {
            const int ia = base + wid + NW * lane;
            if (ia < natoms) {
                my_s = ia + s_roff[(ia >= p1) + (ia >= p2) + (ia >= p3)];
                my_r0 = row_start[my_s];
                my_len = rcache.len[my_s];
            }
        }
        int nrows = (natoms - base - wid + NW - 1) / NW;
        nrows = nrows < 0 ? 0 : (nrows > 32 ? 32 : nrows);
        auto issue = [&](int l) {                               // all lanes call; lane 0 issues
            const int64_t r0 = __shfl_sync(0xffffffffu, my_r0, l);
            const int pl = (__shfl_sync(0xffffffffu, my_len, l) + 31) & ~31;
            if (lane == 0 && pl > 0 && pl <= RCAP) {
                const unsigned bar = smem_u32(&bars[wid][l & 1]);
                const unsigned dst = smem_u32(mybuf + (size_t)(l & 1) * BUFB);
                mbar_expect_tx(bar, (unsigned)pl * 6u);
                bulk_g2s(dst, rcache.t + r0, (unsigned)pl * 4u, bar);
                bulk_g2s(dst + RCAP * 4, rcache.idx + r0, (unsigned)pl * 2u, bar);
            }
        };
        if (nrows > 0) issue(0);
        for (int l = 0; l < nrows; ++l) {
            if (l + 1 < nrows) issue(l + 1);
            const int s = __shfl_sync(0xffffffffu, my_s, l);
            const int len_s = __shfl_sync(0xffffffffu, my_len, l);
            const int padlen = (len_s + 31) & ~31;
            float a3 = 0.f;
            auto term = [&](unsigned e, float v) {
                float qj;
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(qj) : "r"(qs_addr + (SCALED ? e >> 2 : e << 2)));
                a3 = fmaf(qj, v, a3);
            };
            if (padlen > 0 && padlen <= RCAP) {
                const unsigned bar = smem_u32(&bars[wid][l & 1]);
                mbar_wait(bar, (l & 1) ? phase1 : phase0);
                if (l & 1) phase1 ^= 1; else phase0 ^= 1;
                const float4* tv = (const float4*)(mybuf + (size_t)(l & 1) * BUFB);
                const uint2* ev = (const uint2*)(mybuf + (size_t)(l & 1) * BUFB + RCAP * 4);
                for (int c = 4 * lane; c < padlen; c += 128) {
                    const float4 v = tv[c >> 2];
                    const uint2 e = ev[c >> 2];
                    term(e.x & 0xffffu, v.x);
                    term(e.x >> 16, v.y);
                    term(e.y & 0xffffu, v.z);
                    term(e.y >> 16, v.w);
                }
                // the buffer is written again by the copy engine two rows on: order these reads before it
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
            } else if (padlen > 0) {                            // a row longer than the buffer: straight from global
                const int64_t r0 = __shfl_sync(0xffffffffu, my_r0, l);
                for (int c = 4 * lane; c < padlen; c += 128) {
                    const float4 v = __ldg((const float4*)(rcache.t + r0 + c));
                    const uint2 e = __ldg((const uint2*)(rcache.idx + r0 + c));
                    term(e.x & 0xffffu, v.x);
                    term(e.x >> 16, v.y);
                    term(e.y & 0xffffu, v.z);
                    term(e.y >> 16, v.w);
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) a3 += __shfl_xor_sync(0xffffffffu, a3, o);
            if (lane == 0) out[s] = make_float4(0.f, 0.f, 0.f, a3);
        }
    }
}

// ---- batched right-hand sides on the geometry cache (NEXT-1) ------------------------------------------------------
// qs[v][s] = q[v][perm[s]] for v < nvec, zero for nvec <= v < nv (the kernel takes two or four vectors)
__global__ void k_sort_charges_multi(int64_t n, int nvec, int nv, const float* __restrict__ q, const int* __restrict__ perm,
                                     float* __restrict__ qs)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int64_t i = perm[s];
    for (int v = 0; v < nv; ++v) qs[(int64_t)v * n + s] = v < nvec ? q[(int64_t)v * n + i] : 0.f;
}

__global__ void k_multi_to_out(int64_t n, const float* __restrict__ r, float4* __restrict__ out)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s < n) out[s] = make_float4(0.f, 0.f, 0.f, r[s]);
}

// Real-space potentials of nvec (1..4) charge vectors q[nvec][n] (caller order) in one pass over the geometry cache of
// `nl` (which must be warm: the caller checks); results in ctx->batch_r [nv][n], sorted order.
int realspace_cached_multi(sqeq_ctx* ctx, const sqeq_nlist* nl, int nvec, const float* q, cudaStream_t st)
{
    const int64_t n = nl->n;
    const int nv = nvec <= 2 ? 2 : 4;
    SQEQ_TRY(sqeq_reserve(ctx, ctx->batch_q, sizeof(float) * 4 * (size_t)n));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->batch_r, sizeof(float) * 4 * (size_t)n));
    GeomCache& gc = ctx->gc;
    RealCache rcache = {(uint16_t*)gc.idx.p, (float*)gc.t.p, (int*)gc.len.p};
    k_sort_charges_multi<<<ceil_div(n, 256), 256, 0, st>>>(n, nvec, nv, q, nl->perm, (float*)ctx->batch_q.p);
    KERNEL_CHECK(ctx);
    StageTimer tm(ctx, SQEQ_T_REAL, st);
    const int ngroups = nl->gg.ng[0] * nl->gg.ng[1] * nl->gg.ng[2];
    const size_t sm = sizeof(float) * nv * ((size_t)nl->max_pop + 1);
    auto kern = nv == 2 ? (nl->lshift ? k_real_cached_multi<2, true> : k_real_cached_multi<2, false>)
                        : (nl->lshift ? k_real_cached_multi<4, true> : k_real_cached_multi<4, false>);
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    kern<<<ngroups, REAL_NT, sm, st>>>((const float*)ctx->batch_q.p, n, nl->cell_start, nl->gg, nl->row_start, ngroups,
                                       (float*)ctx->batch_r.p, rcache);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

// vector v of the last realspace_cached_multi into the slot the assembly reads
int realspace_multi_select(sqeq_ctx* ctx, const sqeq_nlist* nl, int v, cudaStream_t st)
{
    const int64_t n = nl->n;
    SQEQ_TRY(sqeq_reserve(ctx, ctx->real_out, sizeof(float4) * n));
    k_multi_to_out<<<ceil_div(n, 256), 256, 0, st>>>(n, (const float*)ctx->batch_r.p + (int64_t)v * n, (float4*)ctx->real_out.p);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

// geom: GEOM_NEW = plain evaluation; GEOM_BUILD = plain evaluation that also writes the geometry cache (t, and g
// when want_force); GEOM_REUSE_PHI / GEOM_REUSE_FIELD = potential / field from the cache.  The cache belongs to
// (list, positions of the last prep_atoms, rc, alpha); the drivers that keep the geometry fixed ask for it.
int realspace_run(sqeq_ctx* ctx, const sqeq_nlist* nl, double rc, double alpha, bool want_force,
                  cudaStream_t st, int geom, bool want_phi)
{
    const int64_t n = nl->n;
    SQEQ_TRY(sqeq_reserve(ctx, ctx->real_out, sizeof(float4) * n));
    RealParams p;
    p.Lx = (float)nl->box[0]; p.Ly = (float)nl->box[1]; p.Lz = (float)nl->box[2];
    p.rc2 = (float)(rc * rc);
    p.pa = (float)(ERFC_P * alpha);
    p.c2 = (float)(2.0 * alpha / sqrt(M_PI));
    p.na2l2e = (float)(-alpha * alpha * 1.4426950408889634);
    StageTimer tm(ctx, SQEQ_T_REAL, st);
    const int nb = ceil_div(n * 32, 256);
    if (nl->fmt == 1) {
        const size_t smem = sizeof(float4) * ((size_t)nl->max_pop + 1);
        const int ngroups = nl->gg.ng[0] * nl->gg.ng[1] * nl->gg.ng[2];
        const bool lean = ctx->overlap_now;
        GeomCache& gc = ctx->gc;
        RealCache rcache = {(uint16_t*)gc.idx.p, (float*)gc.t.p, (int*)gc.len.p};
        const bool fixed = geom != GEOM_NEW && !lean;
        const bool hit = fixed && gc.valid && gc.nl == nl && gc.serial == nl->serial && gc.rc == rc && gc.alpha == alpha;
        const uint16_t* list = (const uint16_t*)nl->nbr;
        const int* lens = nl->row_len;
        if (hit && !want_force) {
            // NEXT-1: the potential as a sparse product over the cached t
            const size_t sm = sizeof(float) * ((size_t)nl->max_pop + 1);
            constexpr int RCAP = 512;
            const size_t sm_tma = (size_t)(REAL_NT / 32) * 2 * RCAP * 6 + sm + 128;
            if (ctx->real_tma && nl->max_row <= RCAP && sm_tma <= 113 * 1024) {
                // rows streamed by the bulk-copy engine (two 111 KB blocks per SM)
                auto kern = nl->lshift ? k_real_cached_tma<true, RCAP> : k_real_cached_tma<false, RCAP>;
                CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_tma));
                kern<<<ngroups, REAL_NT, sm_tma, st>>>((const float4*)ctx->xq.p, nl->cell_start, nl->gg, nl->row_start, p, ngroups,
                                                       (float4*)ctx->real_out.p, rcache);
                KERNEL_CHECK(ctx);
                return SQEQ_OK;
            }
            auto kern = nl->lshift ? k_real_cached<0, true> : k_real_cached<0, false>;
            CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            kern<<<ngroups, REAL_NT, sm, st>>>((const float4*)ctx->xq.p, nl->cell_start, nl->gg, nl->row_start, p, ngroups,
                                               (float4*)ctx->real_out.p, rcache);
            KERNEL_CHECK(ctx);
            return SQEQ_OK;
        }
        if (hit) {
            // forces on a cached geometry: the plain kernel over the compact rows (no skin entries)
            list = (const uint16_t*)gc.idx.p;
            lens = (const int*)gc.len.p;
        }
        const bool build = fixed && !hit;
        if (build) {
            // first evaluation on this geometry: also write the compact in-range rows and their t
            SQEQ_TRY(sqeq_reserve(ctx, gc.idx, sizeof(uint16_t) * (size_t)nl->n_slots));
            SQEQ_TRY(sqeq_reserve(ctx, gc.t, sizeof(float) * (size_t)nl->n_slots));
            SQEQ_TRY(sqeq_reserve(ctx, gc.len, sizeof(int) * (size_t)n));
            rcache = {(uint16_t*)gc.idx.p, (float*)gc.t.p, (int*)gc.len.p};
            gc.valid = true; gc.nl = nl; gc.serial = nl->serial; gc.rc = rc; gc.alpha = alpha;
        }
        // beside the PME side stream: a persistent grid of two lean blocks per SM leaves registers and shared
        // memory for one PME block per SM; otherwise one block per group
        auto kern = nl->lshift ? (want_force ? k_real_staged<true, true, false> : k_real_staged<false, true, false>)
                               : (want_force ? k_real_staged<true, false, false> : k_real_staged<false, false, false>);
        if (lean)
            kern = nl->lshift ? (want_force ? k_real_staged<true, true, true> : k_real_staged<false, true, true>)
                              : (want_force ? k_real_staged<true, false, true> : k_real_staged<false, false, true>);
        if (build)
            kern = nl->lshift ? (want_force ? k_real_staged<true, true, false, 1> : k_real_staged<false, true, false, 1>)
                              : (want_force ? k_real_staged<true, false, false, 1> : k_real_staged<false, false, false, 1>);
        const int lean_bps = ctx->real_lean_blocks;
        const int nblocks = lean ? (ngroups < lean_bps * ctx->sm_count ? ngroups : lean_bps * ctx->sm_count) : ngroups;
        CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<nblocks, REAL_NT, smem, st>>>((const float4*)ctx->xq.p, nl->cell_start, nl->gg, nl->row_start, lens,
                                         list, hit ? nullptr : nl->grp_slice, p, ngroups, (float4*)ctx->real_out.p, rcache);
    } else if (want_force)
        k_real<true><<<nb, 256, 0, st>>>(n, (const float4*)ctx->xq.p, nl->row_start, nl->row_len, (const uint32_t*)nl->nbr, p,
                                          (float4*)ctx->real_out.p);
    else
        k_real<false><<<nb, 256, 0, st>>>(n, (const float4*)ctx->xq.p, nl->row_start, nl->row_len, (const uint32_t*)nl->nbr, p,
                                           (float4*)ctx->real_out.p);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

// ------------------------------------------------------------------------------------------------
// a-9: phi_i = phi_real + phi_rec - (2 alpha/sqrt(pi)) q_i ; F = q_i (f_real + f_rec) with f the
// per-unit-charge fields the two kernels leave behind (field != 0: write f itself, used by the
// shadow-MD force of Eq. 20); E = 1/2 sum q phi.  Written back in the caller's atom order.
// scal[0] += E (fp64 accumulation).
template <bool FORCE>
__global__ void k_assemble(int64_t n, const float4* __restrict__ xq, const float4* __restrict__ real_out,
                           const float4* __restrict__ rec_out, const int* __restrict__ perm, float cself,
                           int field, float* __restrict__ phi, float* __restrict__ force,
                           double* __restrict__ scal)
{
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double e = 0.0;
    if (s < n) {
        const float4 a = real_out[s], b = rec_out[s];
        const float qi = xq[s].w;
        const float ph = a.w + b.w - cself * qi;
        const int64_t o = perm[s];
        if (phi) phi[o] = ph;
        if (FORCE) {
            const float sc = field ? 1.f : qi;
            force[3 * o + 0] = sc * (a.x + b.x);
            force[3 * o + 1] = sc * (a.y + b.y);
            force[3 * o + 2] = sc * (a.z + b.z);
        }
        e = 0.5 * (double)qi * (double)ph;
    }
    if (scal) {
        __shared__ double red[8];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e;
        __syncthreads();
        if (threadIdx.x < 8) {
            e = red[threadIdx.x];
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) e += __shfl_xor_sync(0xffu, e, o);
            if (threadIdx.x == 0) atomicAdd(scal, e);
        }
    }
}

int assemble_run(sqeq_ctx* ctx, const sqeq_nlist* nl, double alpha, float* phi, float* force,
                 bool want_energy, bool field_mode, cudaStream_t st)
{
    const int64_t n = nl->n;
    const float cself = (float)(2.0 * alpha / sqrt(M_PI));
    double* scal = want_energy ? (double*)ctx->scal.p : nullptr;
    StageTimer tm(ctx, SQEQ_T_ASSEMBLE, st);
    if (want_energy) CUDA_TRY(ctx, cudaMemsetAsync(ctx->scal.p, 0, sizeof(double), st));
    if (force)
        k_assemble<true><<<ceil_div(n, 256), 256, 0, st>>>(n, (const float4*)ctx->xq.p,
            (const float4*)ctx->real_out.p, (const float4*)ctx->rec_out.p, nl->perm, cself, field_mode ? 1 : 0, phi, force, scal);
    else
        k_assemble<false><<<ceil_div(n, 256), 256, 0, st>>>(n, (const float4*)ctx->xq.p,
            (const float4*)ctx->real_out.p, (const float4*)ctx->rec_out.p, nl->perm, cself, field_mode ? 1 : 0, phi, force, scal);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}
