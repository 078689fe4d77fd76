// nlist.cu -- cell-list neighbour build (section 3.1 / Alg. 1), steps a-1, a-2.
//
// a-1  wrap + bin (fp64 cell index) -> counting sort by cell -> per-cell sort by caller index
//      (deterministic order) -> cell-major float4 positions, permutation, wrap counts.
// a-2  pair enumeration: one warp per atom walks the 27 (cell, image) neighbours; candidates are
//      contiguous float4 runs (coalesced 512 B per warp load); distance test in fp32 on wrapped
//      coordinates with a guard band, inside which the decision is taken by the exact fp64
//      predicate of DESIGN.md R-NL on the raw caller positions (individually rounded IEEE ops, no
//      FMA contraction) -- this is what makes the set bit-identical to the O(N^2) definition.
//      Count pass -> scan -> fill pass; output is a directed CSR, entry = j | shift_code << 27,
//      shift_code = (sx+1)*9 + (sy+1)*3 + (sz+1) with s the periodic image shift in box lengths.
//
// Unlike Alg. 1 there is no [N,27,Cmax] candidate tensor and no padded cells[nx,ny,nz,Cmax].
#include <math.h>

#include "common.cuh"

struct NLGeom {
    double L[3];
    int    nc[3];
    float  Lf[3];
    float  rl2f;
    float  band;
    double rl2;
};

// wrapped coordinate in [0, L] and the integer wrap count w with x = xw + w*L (up to rounding)
__device__ __forceinline__ double wrap_coord(double x, double L, int& w)
{
    double fw = floor(x / L);
    double xw = x - fw * L;
    if (xw < 0.0) { xw += L; fw -= 1.0; }
    if (xw >= L) { xw -= L; fw += 1.0; }
    if (xw < 0.0) xw = 0.0;
    w = (int)fw;
    return xw;
}

__device__ __forceinline__ int cell_index(double xw, double L, int nc)
{
    int c = (int)(xw * (double)nc / L);
    return c >= nc ? nc - 1 : (c < 0 ? 0 : c);
}

__global__ void k_bin(int64_t n, const float* __restrict__ pos, NLGeom g, int* __restrict__ cell_id,
                      int* __restrict__ cell_count, int* __restrict__ flag)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    int c[3];
    bool bad = false;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        float xf = pos[3 * i + d];
        if (!isfinite(xf)) { bad = true; xf = 0.f; }
        int w;
        double xw = wrap_coord((double)xf, g.L[d], w);
        if (w > 127 || w < -127) bad = true;
        c[d] = cell_index(xw, g.L[d], g.nc[d]);
    }
    if (bad) atomicOr(flag, 1);
    int cid = (c[0] * g.nc[1] + c[1]) * g.nc[2] + c[2];
    cell_id[i] = cid;
    atomicAdd(&cell_count[cid], 1);
}

__global__ void k_scatter(int64_t n, const int* __restrict__ cell_id, const int* __restrict__ cell_start,
                          int* __restrict__ cell_fill, int* __restrict__ perm)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    int c = cell_id[i];
    int slot = cell_start[c] + atomicAdd(&cell_fill[c], 1);
    perm[slot] = (int)i;
}

// One block per cell: sort the cell's caller indices ascending (bitonic, shared memory) so that the
// cell-major order -- and with it every later summation order -- does not depend on atomics timing.
#define SORT_CAP 2048
__global__ void k_sort_cells(const int* __restrict__ cell_start, int* __restrict__ perm)
{
    __shared__ int s[SORT_CAP];
    int c = blockIdx.x;
    int beg = cell_start[c], m = cell_start[c + 1] - beg;
    if (m <= 1 || m > SORT_CAP) return;
    int p2 = 1;
    while (p2 < m) p2 <<= 1;
    for (int t = threadIdx.x; t < p2; t += blockDim.x) s[t] = t < m ? perm[beg + t] : 0x7fffffff;
    __syncthreads();
    for (int k = 2; k <= p2; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < p2; t += blockDim.x) {
                int x = t ^ j;
                if (x > t) {
                    int a = s[t], b = s[x];
                    bool up = (t & k) == 0;
                    if ((a > b) == up) { s[t] = b; s[x] = a; }
                }
            }
            __syncthreads();
        }
    for (int t = threadIdx.x; t < m; t += blockDim.x) perm[beg + t] = s[t];
}

__global__ void k_reorder(int64_t n, const float* __restrict__ pos, const int* __restrict__ perm,
                          NLGeom g, float4* __restrict__ xq, int* __restrict__ cell_of,
                          char4* __restrict__ wrapc)
{
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= n) return;
    int o = perm[s];
    float xw[3];
    int w[3], c[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double x = wrap_coord((double)pos[3 * (int64_t)o + d], g.L[d], w[d]);
        c[d] = cell_index(x, g.L[d], g.nc[d]);
        xw[d] = (float)x;
    }
    xq[s] = make_float4(xw[0], xw[1], xw[2], 0.f);
    cell_of[s] = (c[0] * g.nc[1] + c[1]) * g.nc[2] + c[2];
    wrapc[s] = make_char4((signed char)w[0], (signed char)w[1], (signed char)w[2], 0);
}

// ------------------------------------------------------------------------------------------ scan
// exclusive scan, 1024 elements per block, recursive over block sums
template <typename Tin>
__global__ void k_scan_blocks(int64_t n, const Tin* __restrict__ in, int64_t* __restrict__ out,
                              int64_t* __restrict__ block_sums)
{
    __shared__ int64_t warp_tot[32];
    int64_t i = blockIdx.x * (int64_t)1024 + threadIdx.x;
    int64_t v = i < n ? (int64_t)in[i] : 0;
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int64_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int64_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_tot[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int64_t t = warp_tot[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int64_t y = __shfl_up_sync(0xffffffffu, t, o);
            if (lane >= o) t += y;
        }
        warp_tot[lane] = t;
    }
    __syncthreads();
    int64_t off = wid > 0 ? warp_tot[wid - 1] : 0;
    if (i < n) out[i] = off + x - v;
    if (threadIdx.x == 1023 && block_sums) block_sums[blockIdx.x] = off + x;
}

__global__ void k_scan_add(int64_t n, int64_t* __restrict__ out, const int64_t* __restrict__ block_off)
{
    int64_t i = blockIdx.x * (int64_t)1024 + threadIdx.x;
    if (i < n) out[i] += block_off[blockIdx.x];
}

__global__ void k_i64_to_i32(int64_t n, const int64_t* __restrict__ in, int* __restrict__ out)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) out[i] = (int)in[i];
}

// out[0..n] (n+1 entries) = exclusive scan of in[0..n); out[n] = total.  in must have n+1 readable
// entries with in[n] ignored: we scan n+1 elements with a zero tail supplied by the caller.
template <typename Tin>
static int exclusive_scan(sqeq_ctx* ctx, int64_t n1, const Tin* in, int64_t* out, cudaStream_t st)
{
    int nb = ceil_div(n1, 1024);
    int64_t* sums = nullptr;
    if (nb > 1) CUDA_TRY(ctx, cudaMallocAsync((void**)&sums, sizeof(int64_t) * 2 * (size_t)nb, st));
    k_scan_blocks<Tin><<<nb, 1024, 0, st>>>(n1, in, out, sums);
    KERNEL_CHECK(ctx);
    if (nb > 1) {
        int64_t* sums_scan = sums + nb;
        SQEQ_TRY(exclusive_scan<int64_t>(ctx, nb, sums, sums_scan, st));
        k_scan_add<<<nb, 1024, 0, st>>>(n1, out, sums_scan);
        KERNEL_CHECK(ctx);
        CUDA_TRY(ctx, cudaFreeAsync(sums, st));
    }
    return SQEQ_OK;
}

// ------------------------------------------------------------------------------------------ pairs
// The exact predicate (DESIGN.md R-NL): d = pos[b]-pos[a] for caller indices a<b, s = -rint(d/L),
// d += s*L, r2 = (dx*dx + dy*dy) + dz*dz, every operation individually rounded; in range <=> r2 < rl2.
__device__ __noinline__ bool exact_in_range(const float* __restrict__ pos, int oi, int oj,
                                            const NLGeom& g)
{
    int a = oi < oj ? oi : oj, b = oi < oj ? oj : oi;
    double d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double dk = __dsub_rn((double)pos[3 * (int64_t)b + k], (double)pos[3 * (int64_t)a + k]);
        double sk = -rint(__ddiv_rn(dk, g.L[k]));
        d[k] = __dadd_rn(dk, __dmul_rn(sk, g.L[k]));
    }
    double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
    return r2 < g.rl2;
}

template <bool FILL>
__global__ void __launch_bounds__(256)
k_pairs(int64_t n, const float4* __restrict__ xq, const int* __restrict__ cell_of,
        const int* __restrict__ cell_start, const int* __restrict__ perm,
        const float* __restrict__ pos, NLGeom g, int* __restrict__ row_count,
        const int64_t* __restrict__ row_start, uint32_t* __restrict__ nbr, int* __restrict__ max_row)
{
    const int lane = threadIdx.x & 31;
    const int64_t s = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (s >= n) return;
    const float4 xi = xq[s];
    const int c = cell_of[s];
    const int cz = c % g.nc[2], cy = (c / g.nc[2]) % g.nc[1], cx = c / (g.nc[2] * g.nc[1]);
    int count = 0;
    const int64_t base = FILL ? row_start[s] : 0;
    const unsigned lt = (1u << lane) - 1u;
    for (int img = 0; img < 27; ++img) {
        int ox = img / 9 - 1, oy = (img / 3) % 3 - 1, oz = img % 3 - 1;
        int nx = cx + ox, ny = cy + oy, nz = cz + oz;
        // image shift of the neighbour cell (in box lengths): non-zero only where the stencil wraps
        int wx = 0, wy = 0, wz = 0;
        if (nx < 0) { nx += g.nc[0]; wx = -1; } else if (nx >= g.nc[0]) { nx -= g.nc[0]; wx = 1; }
        if (ny < 0) { ny += g.nc[1]; wy = -1; } else if (ny >= g.nc[1]) { ny -= g.nc[1]; wy = 1; }
        if (nz < 0) { nz += g.nc[2]; wz = -1; } else if (nz >= g.nc[2]) { nz -= g.nc[2]; wz = 1; }
        const float sx = wx * g.Lf[0], sy = wy * g.Lf[1], sz = wz * g.Lf[2];
        const uint32_t scode = (uint32_t)((wx + 1) * 9 + (wy + 1) * 3 + (wz + 1));
        const int nc = (nx * g.nc[1] + ny) * g.nc[2] + nz;
        const int beg = cell_start[nc], end = cell_start[nc + 1];
        for (int t0 = beg; t0 < end; t0 += 32) {
            const int t = t0 + lane;
            bool ok = false;
            if (t < end) {
                const float4 xj = xq[t];
                const float dx = (xj.x - xi.x) + sx;
                const float dy = (xj.y - xi.y) + sy;
                const float dz = (xj.z - xi.z) + sz;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                if (r2 < g.rl2f + g.band) {
                    if (r2 < g.rl2f - g.band) ok = !(t == s && scode == 13u);
                    else if (!(t == s)) ok = exact_in_range(pos, perm[s], perm[t], g);
                }
            }
            const unsigned m = __ballot_sync(0xffffffffu, ok);
            if (FILL && ok) nbr[base + count + __popc(m & lt)] = (uint32_t)t | (scode << 27);
            count += __popc(m);
        }
    }
    if (!FILL && lane == 0) {
        row_count[s] = count;
        atomicMax(max_row, count);
    }
}

// ------------------------------------------------------------------------------------------ export
__device__ __forceinline__ void decode_img(uint32_t e, int& t, int& ox, int& oy, int& oz)
{
    t = (int)(e & 0x07ffffffu);
    int img = (int)(e >> 27);
    ox = img / 9 - 1;
    oy = (img / 3) % 3 - 1;
    oz = img % 3 - 1;
}

// counts, per CALLER index, the neighbours with a larger caller index
__global__ void k_export_count(int64_t n, const int64_t* __restrict__ row_start,
                               const uint32_t* __restrict__ nbr, const int* __restrict__ perm,
                               int* __restrict__ cnt_orig)
{
    const int lane = threadIdx.x & 31;
    const int64_t s = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (s >= n) return;
    const int oi = perm[s];
    int c = 0;
    for (int64_t k = row_start[s] + lane; k < row_start[s + 1]; k += 32)
        c += perm[nbr[k] & 0x07ffffffu] > oi;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) cnt_orig[oi] = c;
}

#define EXPORT_CAP 4096
// one block per (sorted) atom: collect upper neighbours, sort by caller index j, write canonical rows
__global__ void __launch_bounds__(256)
k_export_fill(int64_t n, const int64_t* __restrict__ row_start, const uint32_t* __restrict__ nbr,
              const int* __restrict__ perm, const char4* __restrict__ wrapc,
              const int64_t* __restrict__ off_orig, int32_t* __restrict__ out_i,
              int32_t* __restrict__ out_j, int8_t* __restrict__ out_s, int* __restrict__ flag)
{
    __shared__ int key[EXPORT_CAP];
    __shared__ int val[EXPORT_CAP];
    __shared__ int cnt;
    const int64_t s = blockIdx.x;
    const int oi = perm[s];
    const int64_t beg = row_start[s], end = row_start[s + 1];
    const int64_t o0 = off_orig[oi];
    const int m = (int)(off_orig[oi + 1] - o0);
    if (m == 0) return;
    if (m > EXPORT_CAP) { if (threadIdx.x == 0) atomicOr(flag, 2); return; }
    if (threadIdx.x == 0) cnt = 0;
    __syncthreads();
    for (int64_t k = beg + threadIdx.x; k < end; k += blockDim.x) {
        uint32_t e = nbr[k];
        int oj = perm[e & 0x07ffffffu];
        if (oj > oi) {
            int p = atomicAdd(&cnt, 1);
            key[p] = oj;
            val[p] = (int)(k - beg);
        }
    }
    __syncthreads();
    int p2 = 1;
    while (p2 < m) p2 <<= 1;
    for (int t = m + threadIdx.x; t < p2; t += blockDim.x) { key[t] = 0x7fffffff; val[t] = 0; }
    __syncthreads();
    for (int k = 2; k <= p2; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < p2; t += blockDim.x) {
                int x = t ^ j;
                if (x > t) {
                    int a = key[t], b = key[x];
                    bool up = (t & k) == 0;
                    if ((a > b) == up) {
                        key[t] = b; key[x] = a;
                        int va = val[t]; val[t] = val[x]; val[x] = va;
                    }
                }
            }
            __syncthreads();
        }
    const char4 wi = wrapc[s];
    for (int t = threadIdx.x; t < m; t += blockDim.x) {
        uint32_t e = nbr[beg + val[t]];
        int tj, ox, oy, oz;
        decode_img(e, tj, ox, oy, oz);
        const char4 wj = wrapc[tj];
        // image code is relative to wrapped coordinates: x_raw = x_wrapped + w*L, so the shift of the
        // raw pair is code - w_j + w_i  (r_j + s*L - r_i in range)
        out_i[o0 + t] = oi;
        out_j[o0 + t] = key[t];
        out_s[3 * (o0 + t) + 0] = (int8_t)(ox - wj.x + wi.x);
        out_s[3 * (o0 + t) + 1] = (int8_t)(oy - wj.y + wi.y);
        out_s[3 * (o0 + t) + 2] = (int8_t)(oz - wj.z + wi.z);
    }
}

// ------------------------------------------------------------------------------------------ host
static void fill_geom(NLGeom& g, const double box[3], double cutoff)
{
    double lmax = 0;
    for (int d = 0; d < 3; ++d) {
        g.L[d] = box[d];
        g.Lf[d] = (float)box[d];
        int nc = (int)floor(box[d] / (cutoff * (1.0 + 1e-6)));
        g.nc[d] = nc < 1 ? 1 : nc;
        lmax = fmax(lmax, box[d]);
    }
    g.rl2 = cutoff * cutoff;
    g.rl2f = (float)g.rl2;
    // fp32 error of r2 on wrapped coordinates: |delta d| <= 1.5 ulp(L) per axis, so
    // |delta r2| <= 2 sqrt(3) r 1.5 L 2^-23 + 3 r^2 2^-24 ~ 5.2 r L 2^-23; band = 3x that.
    g.band = (float)((16.0 * cutoff * lmax + 8.0 * cutoff * cutoff) * ldexp(1.0, -23));
}

int nl_build_impl(sqeq_ctx* ctx, int64_t n, const float* pos, const double box[3], double cutoff,
                  sqeq_nlist** out)
{
    cudaStream_t st = ctx->stream;
    NLGeom g;
    fill_geom(g, box, cutoff);
    // keep cells from becoming absurdly many for huge dilute boxes: at most ~ n cells + 64
    int64_t ncells = (int64_t)g.nc[0] * g.nc[1] * g.nc[2];
    while (ncells > 4 * n + 64) {
        int dmax = 0;
        for (int d = 1; d < 3; ++d) if (g.nc[d] > g.nc[dmax]) dmax = d;
        g.nc[dmax] = (g.nc[dmax] + 1) / 2;
        ncells = (int64_t)g.nc[0] * g.nc[1] * g.nc[2];
    }
    sqeq_nlist* nl = new sqeq_nlist();
    nl->ctx = ctx;
    nl->n = n;
    nl->cutoff = cutoff;
    for (int d = 0; d < 3; ++d) { nl->box[d] = box[d]; nl->ncell[d] = g.nc[d]; }

    int *cell_id = nullptr, *cell_count = nullptr, *cell_fill = nullptr, *flag = nullptr, *row_count = nullptr;
    int64_t* tmp64 = nullptr;
    auto cleanup = [&](int code) {
        cudaFree(cell_id); cudaFree(cell_count); cudaFree(cell_fill); cudaFree(flag);
        cudaFree(row_count); cudaFree(tmp64);
        if (code != SQEQ_OK) sqeq_nl_free(nl);
        return code;
    };
#define NL_TRY(expr) do { int _r = (expr); if (_r != SQEQ_OK) return cleanup(_r); } while (0)
#define NL_CUDA(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) return cleanup(sqeq_fail(ctx, \
        _e == cudaErrorMemoryAllocation ? SQEQ_ENOMEM : SQEQ_ECUDA, "%s: %s", #expr, cudaGetErrorString(_e))); } while (0)

    NL_CUDA(cudaMalloc((void**)&cell_id, sizeof(int) * n));
    NL_CUDA(cudaMalloc((void**)&cell_count, sizeof(int) * (ncells + 1)));
    NL_CUDA(cudaMalloc((void**)&cell_fill, sizeof(int) * (ncells + 1)));
    NL_CUDA(cudaMalloc((void**)&flag, sizeof(int) * 2));
    NL_CUDA(cudaMalloc((void**)&row_count, sizeof(int) * (n + 1)));
    NL_CUDA(cudaMalloc((void**)&tmp64, sizeof(int64_t) * (ncells + 1)));
    NL_CUDA(cudaMalloc((void**)&nl->perm, sizeof(int) * n));
    NL_CUDA(cudaMalloc((void**)&nl->cell_of, sizeof(int) * n));
    NL_CUDA(cudaMalloc((void**)&nl->cell_start, sizeof(int) * (ncells + 1)));
    NL_CUDA(cudaMalloc((void**)&nl->wrapc, sizeof(char4) * n));
    NL_CUDA(cudaMalloc((void**)&nl->row_start, sizeof(int64_t) * (n + 1)));
    NL_TRY(sqeq_reserve(ctx, ctx->xq, sizeof(float4) * n));
    float4* xq = (float4*)ctx->xq.p;

    const int nb = ceil_div(n, 256);
    {
        StageTimer tm(ctx, SQEQ_T_NL_BIN);
        NL_CUDA(cudaMemsetAsync(cell_count, 0, sizeof(int) * (ncells + 1), st));
        NL_CUDA(cudaMemsetAsync(cell_fill, 0, sizeof(int) * (ncells + 1), st));
        NL_CUDA(cudaMemsetAsync(flag, 0, sizeof(int) * 2, st));
        k_bin<<<nb, 256, 0, st>>>(n, pos, g, cell_id, cell_count, flag);
        ctx->launches++;
        NL_TRY(exclusive_scan<int>(ctx, ncells + 1, cell_count, tmp64, st));
        k_i64_to_i32<<<ceil_div(ncells + 1, 256), 256, 0, st>>>(ncells + 1, tmp64, nl->cell_start);
        ctx->launches++;
        k_scatter<<<nb, 256, 0, st>>>(n, cell_id, nl->cell_start, cell_fill, nl->perm);
        ctx->launches++;
        k_sort_cells<<<(int)ncells, 256, 0, st>>>(nl->cell_start, nl->perm);
        ctx->launches++;
        k_reorder<<<nb, 256, 0, st>>>(n, pos, nl->perm, g, xq, nl->cell_of, nl->wrapc);
        ctx->launches++;
        NL_CUDA(cudaGetLastError());
    }
    int h_flag[2] = {0, 0};
    {
        StageTimer tm(ctx, SQEQ_T_NL_PAIRS);
        int* max_row = flag + 1;
        NL_CUDA(cudaMemsetAsync(row_count, 0, sizeof(int) * (n + 1), st));
        const int nbw = ceil_div(n * 32, 256);
        k_pairs<false><<<nbw, 256, 0, st>>>(n, xq, nl->cell_of, nl->cell_start, nl->perm, pos, g,
                                             row_count, nullptr, nullptr, max_row);
        ctx->launches++;
        NL_TRY(exclusive_scan<int>(ctx, n + 1, row_count, nl->row_start, st));
        int64_t total = 0;
        NL_CUDA(cudaMemcpyAsync(&total, nl->row_start + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        NL_CUDA(cudaMemcpyAsync(h_flag, flag, sizeof(int) * 2, cudaMemcpyDeviceToHost, st));
        NL_CUDA(cudaStreamSynchronize(st));
        if (h_flag[0] & 1)
            return cleanup(sqeq_fail(ctx, SQEQ_EINVAL,
                                     "sqeq_nl_build: a position is non-finite or more than 127 box lengths away"));
        nl->n_directed = total;
        nl->max_row = h_flag[1];
        NL_CUDA(cudaMalloc((void**)&nl->nbr, sizeof(uint32_t) * (size_t)(total > 0 ? total : 1)));
        k_pairs<true><<<nbw, 256, 0, st>>>(n, xq, nl->cell_of, nl->cell_start, nl->perm, pos, g,
                                            nullptr, nl->row_start, nl->nbr, nullptr);
        ctx->launches++;
        NL_CUDA(cudaGetLastError());
    }
    NL_CUDA(cudaStreamSynchronize(st));
    *out = nl;
    cleanup(SQEQ_OK);
    return SQEQ_OK;
#undef NL_TRY
#undef NL_CUDA
}

int nl_export_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, int32_t* oi, int32_t* oj, int8_t* shift3)
{
    cudaStream_t st = ctx->stream;
    const int64_t n = nl->n;
    if (nl->n_directed == 0) return SQEQ_OK;
    int* cnt = nullptr;
    int64_t* off = nullptr;
    int* flag = nullptr;
    CUDA_TRY(ctx, cudaMalloc((void**)&cnt, sizeof(int) * (n + 1)));
    CUDA_TRY(ctx, cudaMalloc((void**)&off, sizeof(int64_t) * (n + 1)));
    CUDA_TRY(ctx, cudaMalloc((void**)&flag, sizeof(int)));
    CUDA_TRY(ctx, cudaMemsetAsync(cnt, 0, sizeof(int) * (n + 1), st));
    CUDA_TRY(ctx, cudaMemsetAsync(flag, 0, sizeof(int), st));
    k_export_count<<<ceil_div(n * 32, 256), 256, 0, st>>>(n, nl->row_start, nl->nbr, nl->perm, cnt);
    KERNEL_CHECK(ctx);
    int r = exclusive_scan<int>(ctx, n + 1, cnt, off, st);
    if (r == SQEQ_OK) {
        k_export_fill<<<(unsigned)n, 256, 0, st>>>(n, nl->row_start, nl->nbr, nl->perm, nl->wrapc, off,
                                                    oi, oj, shift3, flag);
        ctx->launches++;
    }
    int h_flag = 0;
    int64_t total = 0;
    cudaMemcpyAsync(&h_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
    cudaMemcpyAsync(&total, off + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(cnt); cudaFree(off); cudaFree(flag);
    if (r != SQEQ_OK) return r;
    if (e != cudaSuccess) return sqeq_fail(ctx, SQEQ_ECUDA, "sqeq_nl_export: %s", cudaGetErrorString(e));
    if (h_flag & 2) return sqeq_fail(ctx, SQEQ_ECAPACITY, "sqeq_nl_export: a row has more than %d upper neighbours", EXPORT_CAP);
    if (total * 2 != nl->n_directed)
        return sqeq_fail(ctx, SQEQ_ECUDA, "sqeq_nl_export: list is not symmetric (%lld upper entries, %lld directed)",
                         (long long)total, (long long)nl->n_directed);
    return SQEQ_OK;
}
