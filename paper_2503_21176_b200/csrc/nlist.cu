// nlist.cu -- cell-list neighbour build (section 3.1 / Alg. 1), steps a-1, a-2.
//
// a-1  wrap + bin (fp64 cell index) -> counting sort by cell -> per-cell sort by caller index
//      (deterministic order) -> cell-major float4 positions, permutation, wrap counts.
//      Cells have edge >= r_list/2 (stencil half-width w = 2 cells per axis), z fastest in memory.
// a-2  pair enumeration in ONE pass: one warp per atom sweeps the contiguous atom runs of the
//      stencil columns that can reach the cutoff sphere (see k_pairs); the distance test is fp32 on
//      wrapped coordinates with a guard band, inside which the decision is taken by the exact fp64
//      predicate of DESIGN.md R-NL on the raw caller positions (individually rounded IEEE ops, no
//      FMA contraction) -- this is what makes the set bit-identical to the O(N^2) definition.
//      Output: directed rows (row_start, row_len) in one array.  Default format: 16-bit indices into the
//      neighbourhood of the atom's 2x2x2 cell group (cellgroup.cuh; stored << 4 while neighbourhoods have
//      fewer than 4095 atoms), rows padded to multiples of 32 entries, each group's rows in one reserved
//      slice.  Fallback format: entry = j | code << 27, code = (sx+1)*9 + (sy+1)*3 + (sz+1) with s the
//      periodic image shift in box lengths.
//
// Unlike Alg. 1 there is no [N,27,Cmax] candidate tensor and no padded cells[nx,ny,nz,Cmax].
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <type_traits>

#include "common.cuh"
#include "cellgroup.cuh"

struct NLGeom {
    double L[3];
    double rl2;
    int    nc[3];
    int    w[3];      // stencil half-width in cells: ceil(r_list / cell edge), 1 or 2
    float  Lf[3];
    float  a[3];      // cell edge
    float  inva[3];
    float  rl2f;
    float  band;      // guard band of the fp32 distance test
    float  marg;      // safety margin (Angstrom) of the fp32 column pruning
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
    cell_of[s] = c[0] | (c[1] << 10) | (c[2] << 20);      // packed cell coordinates (nc <= 1024 per axis)
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
    if (nb > 1) CUDA_TRY(ctx, cudaMallocFromPoolAsync((void**)&sums, sizeof(int64_t) * 2 * (size_t)nb, ctx->pool, st));
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
// Out of line and fed through a pointer so that the hot loop keeps no fp64 state in registers.
struct NLExact {
    double L[3];
    double rl2;
};

__device__ __noinline__ bool exact_in_range(const float* __restrict__ pos, int oi, int oj,
                                            const NLExact* __restrict__ ex)
{
    int a = oi < oj ? oi : oj, b = oi < oj ? oj : oi;
    double d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double L = ex->L[k];
        double dk = __dsub_rn((double)pos[3 * (int64_t)b + k], (double)pos[3 * (int64_t)a + k]);
        double sk = -rint(__ddiv_rn(dk, L));
        d[k] = __dadd_rn(dk, __dmul_rn(sk, L));
    }
    double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
    return r2 < ex->rl2;
}

// Single-pass pair enumeration.  One block per GROUP of 2x2x2 cells (cellgroup.cuh), one warp per atom
// of the group at a time:
//  0. the block lays out the group's neighbourhood (columns x periodic images = pieces) in shared memory;
//  1. lanes build the atom's SEGMENT list: one lane per (x,y) column of its (2w+1)^2 cell stencil; a
//     column is pruned when its rectangle is farther than r_list from the atom, its z-range is trimmed
//     to the chord of the cutoff sphere, and what is left of each piece is one contiguous run of atoms:
//     a segment (begin, end, image code, local-index offset);
//  2. the warp sweeps the segments 32 candidates at a time (coalesced float4 loads), keeps what the fp32
//     test cannot exclude, compacts with ballot/popc into a per-warp staging row in shared memory, and
//     afterwards settles the candidates inside the guard band by the exact fp64 predicate (rare);
//  3. one atomicAdd on a global cursor reserves the row's slice of `nbr`, the staged row is copied out
//     with coalesced stores, and (row_start, row_len) are recorded.
// LOCAL = true emits 16-bit local indices into the group's neighbourhood (for the shared-memory-staged
// real-space kernel), LOCAL = false 32-bit entries j | image code << 27.
// If the cursor passes `capacity`, a row outgrows the staging row or a neighbourhood outgrows 16 bits,
// the kernel keeps counting and the host re-runs it with the now known sizes / the other format.
#define NL_MAXSEG 96
#define NL_WARPS 8
#ifndef NL_BPS
#define NL_BPS 4
#endif
struct NLCounters {
    unsigned long long cursor;     // list slots handed out (fmt 1 rows are padded to whole warps)
    unsigned long long pairs;      // directed pairs
    int max_row;
    int max_pop;
    int stage_overflow;            // k_pairs_staged: a neighbourhood did not fit the shared memory it was launched with
    int pad_;
    NLExact ex;
};

__device__ __forceinline__ int4 lds_int4(unsigned addr)
{
    int4 v;
    asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float4 lds_float4(unsigned addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

template <bool LOCAL>
__global__ void __launch_bounds__(NL_WARPS * 32, NL_BPS)
k_pairs(const float4* __restrict__ xq, const int* __restrict__ cell_of,
        const int* __restrict__ cell_start, const int* __restrict__ perm,
        const float* __restrict__ pos, NLGeom g, GroupGeom gg, int cap_row, int lshift, int est_row,
        unsigned long long capacity, NLCounters* __restrict__ ctr, int64_t* __restrict__ row_start,
        int* __restrict__ row_len, longlong2* __restrict__ grp_slice, void* __restrict__ nbr_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* shtab = (float4*)smem_raw;                                        // [32] image shift vectors
    GroupPiece* pieces = (GroupPiece*)(smem_raw + 32 * sizeof(float4));       // [GRP_MAXPIECE]
    int4* segs_all = (int4*)(pieces + GRP_MAXPIECE);                          // [NL_WARPS][NL_MAXSEG]
    typedef typename std::conditional<LOCAL, uint16_t, uint32_t>::type entry_t;
    float4* segx_all = (float4*)(segs_all + NL_WARPS * NL_MAXSEG);            // [NL_WARPS][NL_MAXSEG] xi - image shift
    entry_t* stage_all = (entry_t*)(segx_all + NL_WARPS * NL_MAXSEG);          // [NL_WARPS][cap_row] list entries
    __shared__ int s_scratch, s_rbeg[GRP_G * GRP_G], s_rpre[GRP_G * GRP_G + 1];
    __shared__ unsigned long long s_base, s_pairs;      // the block's reserved slice of the list; its pair count
    __shared__ int s_used, s_res, s_maxrow;
    if (threadIdx.x < 32) {
        int img = threadIdx.x < 27 ? threadIdx.x : 13;
        shtab[threadIdx.x] = make_float4((img / 9 - 1) * g.Lf[0], ((img / 3) % 3 - 1) * g.Lf[1],
                                         (img % 3 - 1) * g.Lf[2], 0.f);
    }
    const GroupInfo gi = group_layout(gg, cell_start, blockIdx.x, pieces, &s_scratch);
    // the group's own atoms: ge0*ge1 columns, cells c0z .. c0z+ge2-1 of the zero-image piece
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int r = 0; r < GRP_G * GRP_G; ++r) {
            s_rpre[r] = acc;
            const int ix = r / GRP_G, iy = r % GRP_G;
            if (ix < gi.ge[0] && iy < gi.ge[1]) {
                const int colw = ((gi.c0[0] + ix) * gg.nc[1] + gi.c0[1] + iy) * gg.nc[2] + gi.c0[2];
                const int beg = cell_start[colw];
                s_rbeg[r] = beg;
                acc += cell_start[colw + gi.ge[2]] - beg;
            } else {
                s_rbeg[r] = 0;
            }
        }
        s_rpre[GRP_G * GRP_G] = acc;
        if (LOCAL) atomicMax(&ctr->max_pop, gi.pop);
        // ONE global reservation per block (est_row slots per atom, a multiple of 32): the rows then take
        // their slices with a shared-memory counter.  Per-row reservations on the global cursor -- a third
        // of a million atomics on one address -- were what bounded this kernel.  Rows that do not fit the
        // estimate fall back to the global cursor; unused slots at the end of a slice stay empty.
        s_res = acc * est_row;
        s_base = s_res > 0 ? atomicAdd(&ctr->cursor, (unsigned long long)s_res) : 0ull;
        s_used = 0;
        s_maxrow = 0;
        s_pairs = 0ull;
    }
    __syncthreads();
    const int natoms = s_rpre[GRP_G * GRP_G];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int4* segs = segs_all + wid * NL_MAXSEG;
    float4* segx = segx_all + wid * NL_MAXSEG;
    entry_t* stage = stage_all + (size_t)wid * cap_row;
    const int np_grp = gi.ncol * 3;
    const unsigned lt = (1u << lane) - 1u;
    const float hi_thr = g.rl2f + g.band, lo_thr = g.rl2f - g.band;
    const int ny_st = 2 * gg.w[1] + 1;
    const int ncol_atom = (2 * gg.w[0] + 1) * ny_st;
    const int ncz = gg.nc[2];

    for (int ia = wid; ia < natoms; ia += NL_WARPS) {
        int r = 0;
#pragma unroll
        for (int k = 1; k < GRP_G * GRP_G; ++k) r += (ia >= s_rpre[k]);
        const int s = s_rbeg[r] + (ia - s_rpre[r]);
        const float4 xi = xq[s];
        const int c = cell_of[s];                                  // packed cx | cy << 10 | cz << 20
        const int cx = c & 1023, cy = (c >> 10) & 1023, cz = c >> 20;

        // ---- 1. segments
        int nloc = 0;
        int4 loc0 = make_int4(0, 0, 0, 0), loc1 = loc0, loc2 = loc0;
        if (lane < ncol_atom) {
            const int ox = lane / ny_st - gg.w[0], oy = lane % ny_st - gg.w[1];
            const int ux = cx + ox, uy = cy + oy;
            float dxm = fmaxf(fmaxf((float)ux * g.a[0] - xi.x, xi.x - (float)(ux + 1) * g.a[0]) - g.marg, 0.f);
            float dym = fmaxf(fmaxf((float)uy * g.a[1] - xi.y, xi.y - (float)(uy + 1) * g.a[1]) - g.marg, 0.f);
            if (ox == 0) dxm = 0.f;
            if (oy == 0) dym = 0.f;
            const float rem = hi_thr - (dxm * dxm + dym * dym);
            if (rem > 0.f) {
                const float zr = sqrtf(rem) + g.marg;
                int zlo = (int)floorf((xi.z - zr) * g.inva[2]), zhi = (int)floorf((xi.z + zr) * g.inva[2]);
                zlo = max(zlo, cz - gg.w[2]); zlo = min(zlo, cz);
                zhi = min(zhi, cz + gg.w[2]); zhi = max(zhi, cz);
                const int col = (ux - (gi.c0[0] - gg.w[0])) * gi.ncoly + (uy - (gi.c0[1] - gg.w[1]));
                int uxw = ux, uyw = uy, shx, shy;
                const bool valid = grp_wrap(uxw, gg.nc[0], shx) & grp_wrap(uyw, gg.nc[1], shy);
#pragma unroll
                for (int p = 0; p < 3; ++p) {
                    const GroupPiece pc = pieces[col * 3 + p];
                    const int shz = p - 1;
                    const int a = max(zlo, shz * ncz), b = min(zhi, (shz + 1) * ncz - 1);
                    if (valid && pc.len > 0 && a <= b) {
                        const int colw = (uxw * gg.nc[1] + uyw) * ncz - shz * ncz;
                        const int beg = cell_start[colw + a], end = cell_start[colw + b + 1];
                        if (end > beg) {
                            const int4 v = make_int4(beg, end, pc.code, pc.lbase - pc.gbeg);
                            if (nloc == 0) loc0 = v; else if (nloc == 1) loc1 = v; else loc2 = v;
                            ++nloc;
                        }
                    }
                }
            }
        }
        // slots and candidate offsets of the lane's segments: two warp scans (segments, candidates)
        int incl = nloc, cinc = (loc0.y - loc0.x) + (loc1.y - loc1.x) + (loc2.y - loc2.x);
        const int clen = cinc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o), yc = __shfl_up_sync(0xffffffffu, cinc, o);
            if (lane >= o) { incl += y; cinc += yc; }
        }
        const int nseg = __shfl_sync(0xffffffffu, incl, 31);
        const int total = __shfl_sync(0xffffffffu, cinc, 31);      // candidates of this atom
        __syncwarp();
        {
            // record: x = first atom - first candidate number (t = c + x), y = one past its last candidate
            // number, z = image code, w = local-index offset; segx = xi - image shift
            int at = incl - nloc, cpre = cinc - clen;
            const int4 loc[3] = {loc0, loc1, loc2};
#pragma unroll
            for (int k = 0; k < 3; ++k)
                if (k < nloc) {
                    const float4 sh = shtab[loc[k].z];
                    const int len = loc[k].y - loc[k].x;
                    // (the atom's last segment never ends: lanes past the last candidate stay on it)
                    segs[at] = make_int4(loc[k].x - cpre, at + 1 == nseg ? 0x7fffffff : cpre + len, loc[k].z, loc[k].w);
                    segx[at] = make_float4(xi.x - sh.x, xi.y - sh.y, xi.z - sh.z, 0.f);   // d = xj + shift - xi
                    cpre += len;
                    ++at;
                }
        }
        __syncwarp();

        // ---- 2. sweep over the atom's candidates NUMBERED ACROSS SEGMENTS, 32 per step, so that every step
        // but the last runs with all lanes busy whatever the segment lengths.  A lane keeps the record of
        // the segment its candidate number falls in and moves on when the number passes the segment's end.
        // Every candidate whose fp32 r2 is below rl2 + band is kept; a lane that saw one inside the guard
        // band only raises a flag (xq carries 32 padding entries, so the tail is loaded unclamped and masked).
        int count = 0;
        bool band_seen = false;
        uint32_t self_entry = (uint32_t)s | (13u << 27);
        if (LOCAL) {
            // local index of the atom itself: its column of the group, zero-image piece
            const int col = (cx - (gi.c0[0] - gg.w[0])) * gi.ncoly + (cy - (gi.c0[1] - gg.w[1]));
            const GroupPiece pc = pieces[col * 3 + 1];
            self_entry = (uint32_t)(s + pc.lbase - pc.gbeg);
        }
        if (total > 0) {
            // the lane's current segment record, addressed by its 32-bit shared address (one add per advance)
            unsigned sa = (unsigned)__cvta_generic_to_shared(segs);
            constexpr unsigned SEGX = NL_WARPS * NL_MAXSEG * sizeof(int4);      // segx_all - segs_all, bytes
            int4 cur = lds_int4(sa);
            float4 xs0 = lds_float4(sa + SEGX);
#pragma unroll 2
            for (int c = lane; c - lane < total; c += 32) {
                while (c >= cur.y) {
                    sa += sizeof(int4);
                    cur = lds_int4(sa);
                    xs0 = lds_float4(sa + SEGX);
                }
                const int t = c + cur.x;
                const float4 xj = __ldg(xq + t);
                const float dx = xj.x - xs0.x, dy = xj.y - xs0.y, dz = xj.z - xs0.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                // the entry itself tells the atom from its own zero-image copy
                const uint32_t e = LOCAL ? (uint32_t)(t + cur.w) : ((uint32_t)t | ((uint32_t)cur.z << 27));
                const bool ok = r2 < hi_thr && c < total && e != self_entry;
                band_seen |= ok && r2 >= lo_thr;
                const unsigned m = __ballot_sync(0xffffffffu, ok);
                const int at = min(count + __popc(m & lt), cap_row - 1);   // an overflowing row is re-run anyway
                if (ok) stage[at] = (entry_t)e;
                count += __popc(m);
            }
        }
        __syncwarp();
        // guard band (rare): re-decide the staged candidates inside it with the exact fp64 predicate on
        // the raw caller positions, and compact the staging row in place
        if (__any_sync(0xffffffffu, band_seen) && count <= cap_row) {
            const int oi = perm[s];
            int kept = 0;
            for (int k0 = 0; k0 < count; k0 += 32) {
                const int k = k0 + lane;
                bool ok = k < count;
                entry_t e = 0;
                if (ok) {
                    e = stage[k];
                    int t, code;
                    if (LOCAL) {                                      // local index -> piece -> atom, image
                        int lo = 0, hi = np_grp - 1;
                        while (lo < hi) {
                            const int mid = (lo + hi + 1) >> 1;
                            if (pieces[mid].lbase <= (int)e) lo = mid; else hi = mid - 1;
                        }
                        t = pieces[lo].gbeg + ((int)e - pieces[lo].lbase);
                        code = pieces[lo].code;
                    } else {
                        t = (int)((uint32_t)e & 0x07ffffffu);
                        code = (int)((uint32_t)e >> 27);
                    }
                    const float4 xj = __ldg(xq + t);
                    const float4 sh = shtab[code];
                    const float dx = xj.x - (xi.x - sh.x), dy = xj.y - (xi.y - sh.y), dz = xj.z - (xi.z - sh.z);
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));     // same expression as in the sweep
                    if (r2 >= lo_thr) ok = exact_in_range(pos, oi, perm[t], &ctr->ex);
                }
                const unsigned m = __ballot_sync(0xffffffffu, ok);
                __syncwarp();
                if (ok) stage[kept + __popc(m & lt)] = e;              // kept + rank <= k: never ahead of a reader
                __syncwarp();
                kept += __popc(m);
            }
            count = kept;
        }
        __syncwarp();

        // ---- 3. reserve and copy out
        // a local row is padded to a multiple of 32 slots with the index of the neighbourhood's dummy slot
        // (one past its population: an atom far from everything with charge 0), so that the real-space
        // kernel runs whole warps over it and every row starts on a 64-byte boundary
        const int padn = LOCAL ? (count + 31) & ~31 : count;
        unsigned long long off = 0;
        if (lane == 0) {
            const int old = atomicAdd(&s_used, padn);
            off = old + padn <= s_res ? s_base + (unsigned long long)old
                                      : atomicAdd(&ctr->cursor, (unsigned long long)padn);
            atomicAdd(&s_pairs, (unsigned long long)count);
            atomicMax(&s_maxrow, count);
            row_start[s] = (int64_t)off;
            row_len[s] = count;
        }
        off = __shfl_sync(0xffffffffu, off, 0);
        if (count <= cap_row && off + (unsigned long long)padn <= capacity) {
            if (LOCAL) {
                // pad in the staging row, then move 4 entries per lane (rows and staging rows are 64-byte
                // aligned); the shift is applied to both halves of a word at once (indices < 4096 when shifted)
                if (count + lane < padn) stage[count + lane] = (entry_t)gi.pop;
                __syncwarp();
                const uint32_t keep = lshift ? 0x0fff0fffu : 0xffffffffu;
                const uint2* src = (const uint2*)stage;
                uint2* dst = (uint2*)((entry_t*)nbr_out + off);
                for (int k = lane; 4 * k < padn; k += 32) {
                    uint2 w = src[k];
                    w.x = (w.x & keep) << lshift;
                    w.y = (w.y & keep) << lshift;
                    dst[k] = w;
                }
            } else {
                entry_t* dst = (entry_t*)nbr_out + off;
                for (int k = lane; k < count; k += 32) dst[k] = stage[k];
            }
        }
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (natoms > 0) {
            atomicAdd(&ctr->pairs, s_pairs);
            atomicMax(&ctr->max_row, s_maxrow);
        }
        // where the group's rows are (those that fitted the reservation): the real-space kernel prefetches it
        grp_slice[blockIdx.x] = make_longlong2((long long)s_base, (long long)min(s_used, s_res));
    }
}

// The same enumeration with the group's neighbourhood STAGED IN SHARED MEMORY (as the real-space kernel stages it: every
// run copied with its image shift added), used once a build of the same system has told how large neighbourhoods get.
// A warp takes one atom of the group at a time; lanes test which of the neighbourhood's (x,y) COLUMNS can reach the
// cutoff sphere; the surviving columns of one x-row are neighbours in the staged order, so the warp sweeps at most
// (g + 2w) contiguous stretches of the staged array, 32 candidates per step, with conflict-free 16-byte shared loads: no
// per-candidate global load, no segment records, no index arithmetic beyond an add -- half the instructions of k_pairs
// per candidate step and 15 % more candidates (whole columns instead of chords).  The local index a candidate is
// stored under IS its position in the staged array.  Everything after the sweep (guard band settled by the exact
// fp64 predicate, padding, reservation, copy-out) is k_pairs' code.
#define NLS_WARPS 16
#ifndef NLS_BPS
#define NLS_BPS 2
#endif
__global__ void __launch_bounds__(NLS_WARPS * 32, NLS_BPS)
k_pairs_staged(const float4* __restrict__ xq, const int* __restrict__ cell_of, const int* __restrict__ cell_start,
               const int* __restrict__ perm, const float* __restrict__ pos, NLGeom g, GroupGeom gg, int cap_row, int lshift,
               int est_row, int stage_cap, unsigned long long capacity, NLCounters* __restrict__ ctr,
               int64_t* __restrict__ row_start, int* __restrict__ row_len, longlong2* __restrict__ grp_slice,
               uint16_t* __restrict__ nbr_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* xs = (float4*)smem_raw;                                                   // [stage_cap + 33] (32 of slack)
    uint16_t* stage_all = (uint16_t*)(xs + stage_cap + 33);                           // [NLS_WARPS][cap_row]
    __shared__ GroupPiece pieces[GRP_MAXPIECE];
    __shared__ int s_colbeg[GRP_MAXCOL + 1];
    __shared__ int s_scratch, s_rbeg[GRP_G * GRP_G], s_rpre[GRP_G * GRP_G + 1];
    __shared__ unsigned long long s_base, s_pairs;
    __shared__ int s_used, s_res, s_maxrow;
    const GroupInfo gi = group_layout(gg, cell_start, blockIdx.x, pieces, &s_scratch);
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int r = 0; r < GRP_G * GRP_G; ++r) {
            s_rpre[r] = acc;
            const int ix = r / GRP_G, iy = r % GRP_G;
            if (ix < gi.ge[0] && iy < gi.ge[1]) {
                const int colw = ((gi.c0[0] + ix) * gg.nc[1] + gi.c0[1] + iy) * gg.nc[2] + gi.c0[2];
                const int beg = cell_start[colw];
                s_rbeg[r] = beg;
                acc += cell_start[colw + gi.ge[2]] - beg;
            } else {
                s_rbeg[r] = 0;
            }
        }
        s_rpre[GRP_G * GRP_G] = acc;
        atomicMax(&ctr->max_pop, gi.pop);
        if (gi.pop > stage_cap) atomicExch(&ctr->stage_overflow, 1);
        s_res = gi.pop > stage_cap ? 0 : acc * est_row;
        s_base = s_res > 0 ? atomicAdd(&ctr->cursor, (unsigned long long)s_res) : 0ull;
        s_used = 0;
        s_maxrow = 0;
        s_pairs = 0ull;
    }
    // staged start of every column (its three image runs are consecutive in the staged order)
    if (threadIdx.x <= gi.ncol) s_colbeg[threadIdx.x] = threadIdx.x < gi.ncol ? pieces[threadIdx.x * 3].lbase : gi.pop;
    if (gi.pop > stage_cap) {                       // the host re-runs the build with k_pairs
        if (threadIdx.x == 0) grp_slice[blockIdx.x] = make_longlong2(0, 0);
        return;
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int np_grp = gi.ncol * 3;
    for (int ip = wid; ip < np_grp; ip += NLS_WARPS) {
        const GroupPiece pc = pieces[ip];
        if (pc.len == 0) continue;
        const float sx = (pc.code / 9 - 1) * g.Lf[0], sy = ((pc.code / 3) % 3 - 1) * g.Lf[1], sz = (pc.code % 3 - 1) * g.Lf[2];
        for (int k = lane; k < pc.len; k += 32) {
            float4 v = __ldg(xq + pc.gbeg + k);
            v.x += sx; v.y += sy; v.z += sz;
            xs[pc.lbase + k] = v;
        }
    }
    __syncthreads();
    const int natoms = s_rpre[GRP_G * GRP_G];
    uint16_t* stage = stage_all + (size_t)wid * cap_row;
    const unsigned lt = (1u << lane) - 1u;
    const float hi_thr = g.rl2f + g.band, lo_thr = g.rl2f - g.band;
    const unsigned xs_addr = (unsigned)__cvta_generic_to_shared(xs);
    const int ncolx = gi.ncol / gi.ncoly;

    for (int ia = wid; ia < natoms; ia += NLS_WARPS) {
        int r = 0;
#pragma unroll
        for (int k = 1; k < GRP_G * GRP_G; ++k) r += (ia >= s_rpre[k]);
        const int s = s_rbeg[r] + (ia - s_rpre[r]);
        const float4 xi = xq[s];
        const int c = cell_of[s];
        const int cx = c & 1023, cy = (c >> 10) & 1023;
        // the atom's own place in the staged array: its column of the group, zero-image run
        int self_local;
        {
            const int col = (cx - (gi.c0[0] - gg.w[0])) * gi.ncoly + (cy - (gi.c0[1] - gg.w[1]));
            const GroupPiece pc = pieces[col * 3 + 1];
            self_local = s + pc.lbase - pc.gbeg;
        }
        // lane <-> x-row of columns (<= 6): the y-interval of columns whose rectangle is within reach
        int rb = 0, re = 0;                       // staged stretch [rb, re) of this lane's x-row
        if (lane < ncolx) {
            const int ux = gi.c0[0] - gg.w[0] + lane;
            float dxm = fmaxf(fmaxf((float)ux * g.a[0] - xi.x, xi.x - (float)(ux + 1) * g.a[0]) - g.marg, 0.f);
            if (ux == cx) dxm = 0.f;
            const float rem = hi_thr - dxm * dxm;
            if (rem > 0.f && abs(ux - cx) <= gg.w[0]) {
                const float yr = sqrtf(rem) + g.marg;
                int ylo = (int)floorf((xi.y - yr) * g.inva[1]), yhi = (int)floorf((xi.y + yr) * g.inva[1]);
                ylo = max(ylo, cy - gg.w[1]); ylo = min(ylo, cy);
                yhi = min(yhi, cy + gg.w[1]); yhi = max(yhi, cy);
                const int y0 = gi.c0[1] - gg.w[1];
                rb = s_colbeg[lane * gi.ncoly + (ylo - y0)];
                re = s_colbeg[lane * gi.ncoly + (yhi - y0) + 1];
            }
        }
        int count = 0;
        float r2max = 0.f;                         // largest accepted r2: tells whether anything fell into the guard band
        const unsigned self_addr = xs_addr + ((unsigned)self_local << 4);
        for (int xr = 0; xr < ncolx; ++xr) {
            const int beg = __shfl_sync(0xffffffffu, rb, xr), end = __shfl_sync(0xffffffffu, re, xr);
            // the lane's candidate by its shared-memory address (one add per step); the staged array has 32 slots of
            // slack behind it, so the last step of a stretch reads past `end` unclamped and is masked
            unsigned a = xs_addr + ((unsigned)(beg + lane) << 4);
            const unsigned a_end = xs_addr + ((unsigned)end << 4);
#pragma unroll 2
            for (int k0 = beg; k0 < end; k0 += 32, a += 512u) {
                float4 v;
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
                const float dx = v.x - xi.x, dy = v.y - xi.y, dz = v.z - xi.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                const bool ok = r2 < hi_thr && a < a_end && a != self_addr;
                r2max = fmaxf(r2max, ok ? r2 : 0.f);
                const unsigned m = __ballot_sync(0xffffffffu, ok);
                const int at = min(count + __popc(m & lt), cap_row - 1);   // an overflowing row is re-run anyway
                if (ok) stage[at] = (uint16_t)((a - xs_addr) >> 4);
                count += __popc(m);
            }
        }
        const bool band_seen = r2max >= lo_thr;
        __syncwarp();
        // guard band (rare): re-decide the staged candidates inside it with the exact fp64 predicate on the raw
        // caller positions, and compact the staging row in place
        if (__any_sync(0xffffffffu, band_seen) && count <= cap_row) {
            const int oi = perm[s];
            int kept = 0;
            for (int k0 = 0; k0 < count; k0 += 32) {
                const int k = k0 + lane;
                bool ok = k < count;
                uint16_t e = 0;
                if (ok) {
                    e = stage[k];
                    const float4 v = xs[e];
                    const float dx = v.x - xi.x, dy = v.y - xi.y, dz = v.z - xi.z;
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));     // same expression as in the sweep
                    if (r2 >= lo_thr) {
                        int lo = 0, hi = np_grp - 1;                          // local index -> run -> atom
                        while (lo < hi) {
                            const int mid = (lo + hi + 1) >> 1;
                            if (pieces[mid].lbase <= (int)e) lo = mid; else hi = mid - 1;
                        }
                        const int t = pieces[lo].gbeg + ((int)e - pieces[lo].lbase);
                        ok = exact_in_range(pos, oi, perm[t], &ctr->ex);
                    }
                }
                const unsigned m = __ballot_sync(0xffffffffu, ok);
                __syncwarp();
                if (ok) stage[kept + __popc(m & lt)] = e;
                __syncwarp();
                kept += __popc(m);
            }
            count = kept;
        }
        __syncwarp();
        // reserve and copy out (as in k_pairs)
        const int padn = (count + 31) & ~31;
        unsigned long long off = 0;
        if (lane == 0) {
            const int old = atomicAdd(&s_used, padn);
            off = old + padn <= s_res ? s_base + (unsigned long long)old
                                      : atomicAdd(&ctr->cursor, (unsigned long long)padn);
            atomicAdd(&s_pairs, (unsigned long long)count);
            atomicMax(&s_maxrow, count);
            row_start[s] = (int64_t)off;
            row_len[s] = count;
        }
        off = __shfl_sync(0xffffffffu, off, 0);
        if (count <= cap_row && off + (unsigned long long)padn <= capacity) {
            if (count + lane < padn) stage[count + lane] = (uint16_t)gi.pop;
            __syncwarp();
            const uint32_t keep = lshift ? 0x0fff0fffu : 0xffffffffu;
            const uint2* src = (const uint2*)stage;
            uint2* dst = (uint2*)(nbr_out + off);
            for (int k = lane; 4 * k < padn; k += 32) {
                uint2 w = src[k];
                w.x = (w.x & keep) << lshift;
                w.y = (w.y & keep) << lshift;
                dst[k] = w;
            }
        } else if (lane == 0) {
            row_len[s] = 0;                        // never leave a row that points outside the allocation
        }
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (natoms > 0) {
            atomicAdd(&ctr->pairs, s_pairs);
            atomicMax(&ctr->max_row, s_maxrow);
        }
        grp_slice[blockIdx.x] = make_longlong2((long long)s_base, (long long)min(s_used, s_res));
    }
}

// Expands a 16-bit local list to 32-bit entries j | image code << 27 with the same row offsets (used by
// the canonical export only): one block per group, binary search of each entry in the piece table.
__global__ void __launch_bounds__(256)
k_local_to_global(const int* __restrict__ cell_start, GroupGeom gg, const int64_t* __restrict__ row_start,
                  const int* __restrict__ row_len, const uint16_t* __restrict__ nbr16, int lshift,
                  uint32_t* __restrict__ nbr32)
{
    __shared__ GroupPiece pieces[GRP_MAXPIECE];
    __shared__ int s_scratch;
    const GroupInfo gi = group_layout(gg, cell_start, blockIdx.x, pieces, &s_scratch);
    const int np = gi.ncol * 3;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int ix = 0; ix < gi.ge[0]; ++ix)
        for (int iy = 0; iy < gi.ge[1]; ++iy) {
            const int colw = ((gi.c0[0] + ix) * gg.nc[1] + gi.c0[1] + iy) * gg.nc[2] + gi.c0[2];
            const int beg = cell_start[colw], end = cell_start[colw + gi.ge[2]];
            for (int s = beg + wid; s < end; s += 8) {
                const int64_t r0 = row_start[s];
                const int len = row_len[s];
                for (int k = lane; k < len; k += 32) {
                    const int e = nbr16[r0 + k] >> lshift;
                    int lo = 0, hi = np - 1;                 // last piece with lbase <= e
                    while (lo < hi) {
                        const int mid = (lo + hi + 1) >> 1;
                        if (pieces[mid].lbase <= e) lo = mid; else hi = mid - 1;
                    }
                    const GroupPiece pc = pieces[lo];
                    nbr32[r0 + k] = (uint32_t)(pc.gbeg + (e - pc.lbase)) | ((uint32_t)pc.code << 27);
                }
            }
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
                               const int* __restrict__ row_len,
                               const uint32_t* __restrict__ nbr, const int* __restrict__ perm,
                               int* __restrict__ cnt_orig)
{
    const int lane = threadIdx.x & 31;
    const int64_t s = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (s >= n) return;
    const int oi = perm[s];
    int c = 0;
    const int64_t beg = row_start[s], end = beg + row_len[s];
    for (int64_t k = beg + lane; k < end; k += 32)
        c += perm[nbr[k] & 0x07ffffffu] > oi;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) cnt_orig[oi] = c;
}

#define EXPORT_CAP 4096
// one block per (sorted) atom: collect upper neighbours, sort by caller index j, write canonical rows
__global__ void __launch_bounds__(256)
k_export_fill(int64_t n, const int64_t* __restrict__ row_start, const int* __restrict__ row_len,
              const uint32_t* __restrict__ nbr,
              const int* __restrict__ perm, const char4* __restrict__ wrapc,
              const int64_t* __restrict__ off_orig, int32_t* __restrict__ out_i,
              int32_t* __restrict__ out_j, int8_t* __restrict__ out_s, int* __restrict__ flag)
{
    __shared__ int key[EXPORT_CAP];
    __shared__ int val[EXPORT_CAP];
    __shared__ int cnt;
    const int64_t s = blockIdx.x;
    const int oi = perm[s];
    const int64_t beg = row_start[s], end = beg + row_len[s];
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

// Directed rows in the caller's numbering (the paper's two output formats):
// one block per sorted atom collects ALL its neighbours, sorts them by caller index and writes either row oi of an
// ELLPACK matrix [n][K] (padded with -1) or its stretch of a directed COO list (offsets from a scan of the row
// lengths in caller order).  shift = image shift of the ordered pair (oi, oj) on the raw caller positions.
#define EXPORT_ROW_CAP 8192
__global__ void __launch_bounds__(256)
k_export_rows(const int64_t* __restrict__ row_start, const int* __restrict__ row_len, const uint32_t* __restrict__ nbr,
              const int* __restrict__ perm, const char4* __restrict__ wrapc, int K, const int64_t* __restrict__ off_orig,
              int32_t* __restrict__ out_i, int32_t* __restrict__ out_j, int8_t* __restrict__ out_s, int32_t* __restrict__ counts)
{
    extern __shared__ int sh_rows[];
    int* key = sh_rows;
    int* val = sh_rows + EXPORT_ROW_CAP;
    const int64_t s = blockIdx.x;
    const int oi = perm[s];
    const int64_t beg = row_start[s];
    const int m = row_len[s];
    if (counts && threadIdx.x == 0) counts[oi] = m;
    int p2 = 1;
    while (p2 < m) p2 <<= 1;
    for (int t = threadIdx.x; t < p2; t += blockDim.x) {
        key[t] = t < m ? perm[nbr[beg + t] & 0x07ffffffu] : 0x7fffffff;
        val[t] = t;
    }
    __syncthreads();
    for (int k = 2; k <= p2; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < p2; t += blockDim.x) {
                const int x = t ^ j;
                if (x > t) {
                    const int a = key[t], b = key[x];
                    const bool up = (t & k) == 0;
                    if ((a > b) == up) {
                        key[t] = b; key[x] = a;
                        const int va = val[t]; val[t] = val[x]; val[x] = va;
                    }
                }
            }
            __syncthreads();
        }
    const char4 wi = wrapc[s];
    const int64_t o0 = off_orig ? off_orig[oi] : (int64_t)oi * K;
    for (int t = threadIdx.x; t < m; t += blockDim.x) {
        const uint32_t e = nbr[beg + val[t]];
        int tj, ox, oy, oz;
        decode_img(e, tj, ox, oy, oz);
        const char4 wj = wrapc[tj];
        if (out_i) out_i[o0 + t] = oi;
        out_j[o0 + t] = key[t];
        out_s[3 * (o0 + t) + 0] = (int8_t)(ox - wj.x + wi.x);
        out_s[3 * (o0 + t) + 1] = (int8_t)(oy - wj.y + wi.y);
        out_s[3 * (o0 + t) + 2] = (int8_t)(oz - wj.z + wi.z);
    }
    if (!off_orig)
        for (int t = m + threadIdx.x; t < K; t += blockDim.x) {
            out_j[o0 + t] = -1;
            out_s[3 * (o0 + t) + 0] = 0; out_s[3 * (o0 + t) + 1] = 0; out_s[3 * (o0 + t) + 2] = 0;
        }
}

__global__ void k_row_len_orig(int64_t n, const int* __restrict__ row_len, const int* __restrict__ perm, int* __restrict__ cnt)
{
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s < n) cnt[perm[s]] = row_len[s];
}

// ------------------------------------------------------------------------------------------ host
static void fill_geom(NLGeom& g, const double box[3], double cutoff, int64_t n)
{
    double lmax = 0;
    const double rl = cutoff * (1.0 + 1e-6);
    for (int d = 0; d < 3; ++d) {
        g.L[d] = box[d];
        g.Lf[d] = (float)box[d];
        int nc = (int)floor(2.0 * box[d] / rl);          // edge >= r_list/2
        g.nc[d] = nc < 1 ? 1 : (nc > 1024 ? 1024 : nc);
        lmax = fmax(lmax, box[d]);
    }
    // keep cells from becoming absurdly many for huge dilute boxes: at most ~ 4n cells + 64
    while ((int64_t)g.nc[0] * g.nc[1] * g.nc[2] > 4 * n + 64) {
        int dmax = 0;
        for (int d = 1; d < 3; ++d) if (g.nc[d] > g.nc[dmax]) dmax = d;
        g.nc[dmax] = (g.nc[dmax] + 1) / 2;
    }
    for (int d = 0; d < 3; ++d) {
        const double a = box[d] / g.nc[d];
        g.a[d] = (float)a;
        g.inva[d] = (float)(1.0 / a);
        g.w[d] = a >= rl ? 1 : 2;
    }
    g.rl2 = cutoff * cutoff;
    g.rl2f = (float)g.rl2;
    // fp32 error of r2 on wrapped coordinates: |delta d| <= 1.5 ulp(L) per axis, so
    // |delta r2| <= 2 sqrt(3) r 1.5 L 2^-23 + 3 r^2 2^-24 ~ 5.2 r L 2^-23; band = 3x that.
    g.band = (float)((16.0 * cutoff * lmax + 8.0 * cutoff * cutoff) * ldexp(1.0, -23));
    // column pruning compares fp32 cell faces (index * edge) with fp32 wrapped coordinates: both are
    // within a few ulp(L) of the fp64 values the binning used; 64 ulp(L) + 1e-4 of an edge is safe.
    g.marg = (float)(64.0 * lmax * ldexp(1.0, -23) + 1e-4 * lmax / 64.0);
}

static int pool_alloc(sqeq_ctx* ctx, void** p, size_t bytes)
{
    cudaError_t e = cudaMallocFromPoolAsync(p, bytes > 0 ? bytes : 4, ctx->pool, ctx->stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        *p = nullptr;
        return sqeq_fail(ctx, e == cudaErrorMemoryAllocation ? SQEQ_ENOMEM : SQEQ_ECUDA,
                         "neighbour-list allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
    }
    return SQEQ_OK;
}

// stream-ordered frees: safe after every evaluation already enqueued; the handle itself stays
void nl_release_storage(sqeq_nlist* nl)
{
    cudaStream_t st = nl->ctx->stream;
    void** ptrs[] = {(void**)&nl->perm, (void**)&nl->cell_of, (void**)&nl->cell_start, (void**)&nl->wrapc, (void**)&nl->row_start,
                     (void**)&nl->row_len, (void**)&nl->grp_slice, (void**)&nl->pos0, &nl->nbr};
    for (void** p : ptrs) {
        if (*p) cudaFreeAsync(*p, st);
        *p = nullptr;
    }
}

void nl_release(sqeq_nlist* nl)
{
    sqeq_ctx* ctx = nl->ctx;
    nl_release_storage(nl);
    for (size_t k = 0; k < ctx->lists.size(); ++k)
        if (ctx->lists[k] == nl) { ctx->lists[k] = ctx->lists.back(); ctx->lists.pop_back(); break; }
    delete nl;
}

static void fill_group_geom(GroupGeom& gg, const NLGeom& g)
{
    for (int d = 0; d < 3; ++d) {
        gg.nc[d] = g.nc[d];
        gg.ng[d] = (g.nc[d] + GRP_G - 1) / GRP_G;
        gg.w[d] = g.w[d];
    }
}

static size_t pairs_smem(int cap_row, bool local)
{
    return 32 * sizeof(float4) + GRP_MAXPIECE * sizeof(GroupPiece) + (size_t)NL_WARPS * NL_MAXSEG * (sizeof(int4) + sizeof(float4)) +
           (size_t)NL_WARPS * cap_row * (local ? sizeof(uint16_t) : sizeof(uint32_t));
}

static int launch_pairs(sqeq_ctx* ctx, sqeq_nlist* nl, const float* pos, const NLGeom& g, bool local,
                        int lshift, int est_row, int cap_row, size_t capacity, NLCounters* ctr, cudaStream_t st,
                        int stage_cap)
{
    const size_t smem = pairs_smem(cap_row, local);
    const int ngroups = nl->gg.ng[0] * nl->gg.ng[1] * nl->gg.ng[2];
    if (local && stage_cap > 0) {
        // neighbourhoods of known size: candidates from shared memory
        const size_t sm = sizeof(float4) * ((size_t)stage_cap + 33) + (size_t)NLS_WARPS * cap_row * sizeof(uint16_t);
        CUDA_TRY(ctx, cudaFuncSetAttribute(k_pairs_staged, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        k_pairs_staged<<<ngroups, NLS_WARPS * 32, sm, st>>>((const float4*)ctx->xq.p, nl->cell_of, nl->cell_start, nl->perm, pos, g,
            nl->gg, cap_row, lshift, est_row, stage_cap, (unsigned long long)capacity, ctr, nl->row_start, nl->row_len, nl->grp_slice,
            (uint16_t*)nl->nbr);
        KERNEL_CHECK(ctx);
        return SQEQ_OK;
    }
    if (local) {
        CUDA_TRY(ctx, cudaFuncSetAttribute(k_pairs<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        k_pairs<true><<<ngroups, NL_WARPS * 32, smem, st>>>((const float4*)ctx->xq.p, nl->cell_of, nl->cell_start,
            nl->perm, pos, g, nl->gg, cap_row, lshift, est_row, (unsigned long long)capacity, ctr, nl->row_start, nl->row_len, nl->grp_slice, nl->nbr);
    } else {
        CUDA_TRY(ctx, cudaFuncSetAttribute(k_pairs<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        k_pairs<false><<<ngroups, NL_WARPS * 32, smem, st>>>((const float4*)ctx->xq.p, nl->cell_of, nl->cell_start,
            nl->perm, pos, g, nl->gg, cap_row, lshift, est_row, (unsigned long long)capacity, ctr, nl->row_start, nl->row_len, nl->grp_slice, nl->nbr);
    }
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

int nl_build_impl(sqeq_ctx* ctx, int64_t n, const float* pos, const double box[3], double cutoff,
                  sqeq_nlist** out)
{
    cudaStream_t st = ctx->stream;
    NLGeom g;
    fill_geom(g, box, cutoff, n);
    const int64_t ncells = (int64_t)g.nc[0] * g.nc[1] * g.nc[2];
    sqeq_nlist* nl = new sqeq_nlist();
    nl->ctx = ctx;
    nl->serial = ++ctx->nl_serial;
    nl->n = n;
    nl->cutoff = cutoff;
    for (int d = 0; d < 3; ++d) { nl->box[d] = box[d]; nl->ncell[d] = g.nc[d]; }
    fill_group_geom(nl->gg, g);

    int *cell_id = nullptr, *cell_count = nullptr, *cell_fill = nullptr, *flag = nullptr;
    int64_t* tmp64 = nullptr;
    NLCounters* ctr = nullptr;
    auto cleanup = [&](int code) {
        void* tmp[] = {cell_id, cell_count, cell_fill, flag, tmp64, ctr};
        for (void* p : tmp) if (p) cudaFreeAsync(p, st);
        if (code != SQEQ_OK) { nl_release_storage(nl); delete nl; }
        return code;
    };
#define NL_TRY(expr) do { int _r = (expr); if (_r != SQEQ_OK) return cleanup(_r); } while (0)
#define NL_CUDA(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) return cleanup(sqeq_fail(ctx, \
        _e == cudaErrorMemoryAllocation ? SQEQ_ENOMEM : SQEQ_ECUDA, "%s: %s", #expr, cudaGetErrorString(_e))); } while (0)

    NL_TRY(pool_alloc(ctx, (void**)&cell_id, sizeof(int) * n));
    NL_TRY(pool_alloc(ctx, (void**)&cell_count, sizeof(int) * (ncells + 1)));
    NL_TRY(pool_alloc(ctx, (void**)&cell_fill, sizeof(int) * (ncells + 1)));
    NL_TRY(pool_alloc(ctx, (void**)&flag, sizeof(int) * 2));
    NL_TRY(pool_alloc(ctx, (void**)&tmp64, sizeof(int64_t) * (ncells + 1)));
    NL_TRY(pool_alloc(ctx, (void**)&ctr, sizeof(NLCounters)));
    NL_TRY(pool_alloc(ctx, (void**)&nl->perm, sizeof(int) * n));
    NL_TRY(pool_alloc(ctx, (void**)&nl->cell_of, sizeof(int) * n));
    NL_TRY(pool_alloc(ctx, (void**)&nl->cell_start, sizeof(int) * (ncells + 1)));
    NL_TRY(pool_alloc(ctx, (void**)&nl->wrapc, sizeof(char4) * n));
    NL_TRY(pool_alloc(ctx, (void**)&nl->row_start, sizeof(int64_t) * n));
    NL_TRY(pool_alloc(ctx, (void**)&nl->row_len, sizeof(int) * n));
    NL_TRY(pool_alloc(ctx, (void**)&nl->pos0, sizeof(float) * 3 * n));
    NL_TRY(pool_alloc(ctx, (void**)&nl->grp_slice, sizeof(longlong2) * (size_t)nl->gg.ng[0] * nl->gg.ng[1] * nl->gg.ng[2]));
    ctx->gc.valid = false;             // the build reuses ctx->xq: any prepared geometry is gone
    ctx->geom_serial++;
    NL_TRY(sqeq_reserve(ctx, ctx->xq, sizeof(float4) * (n + 32)));     // 32 padding entries: see k_pairs
    float4* xq = (float4*)ctx->xq.p;
    NL_CUDA(cudaMemsetAsync(xq + n, 0x7f, sizeof(float4) * 32, st));    // 3.4e38: far from everything

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
        // per-cell sort: block size from the mean occupancy (cells hold ~10 atoms at liquid density)
        int sort_threads = 32;
        while (sort_threads < 256 && sort_threads < 2 * n / ncells) sort_threads <<= 1;
        k_sort_cells<<<(int)ncells, sort_threads, 0, st>>>(nl->cell_start, nl->perm);
        ctx->launches++;
        k_reorder<<<nb, 256, 0, st>>>(n, pos, nl->perm, g, xq, nl->cell_of, nl->wrapc);
        ctx->launches++;
        NL_CUDA(cudaMemcpyAsync(nl->pos0, pos, sizeof(float) * 3 * n, cudaMemcpyDeviceToDevice, st));   // for sqeq_nl_max_drift
        NL_CUDA(cudaGetLastError());
    }
    {
        StageTimer tm(ctx, SQEQ_T_NL_PAIRS);
        // sizes: from the previous build of the same system if there was one, else from the mean
        // density; the kernel reports the exact sizes and is re-run if either estimate was short
        const double vol = box[0] * box[1] * box[2];
        const double mean_row = 4.0 / 3.0 * M_PI * cutoff * cutoff * cutoff * (double)n / vol;
        size_t capacity;
        int cap_row;
        int est_row;                   // slots a block reserves per atom (k_pairs), a multiple of 32
        if (ctx->nl_last_n == n && ctx->nl_last_total > 0) {
            capacity = (size_t)(1.08 * (double)ctx->nl_last_total) + 4096;
            cap_row = (int)(1.2 * ctx->nl_last_max_row) + 32;
            est_row = (int)(1.06 * (double)ctx->nl_last_pairs / (double)n) + 32;
        } else {
            capacity = (size_t)(1.3 * mean_row * (double)n) + 128 * (size_t)n + 4096;
            cap_row = (int)(1.5 * mean_row) + 128;
            est_row = (int)(1.1 * mean_row) + 48;
        }
        est_row = (est_row + 31) & ~31;
        cap_row = (cap_row + 31) & ~31;
        NLCounters* h = (NLCounters*)ctx->h_nl;                    // pinned: result, init image, bin flag
        NLCounters* hinit = h + 1;
        int* h_flag = (int*)(h + 2);
        // entry format: 16-bit local indices for the shared-memory-staged real-space kernel unless a
        // group's neighbourhood is too populous for 16 bits / shared memory (or SQEQ_REAL_STAGED=0)
        bool local = !ctx->real_staged_off && !(ctx->nl_last_n == n && ctx->nl_last_fmt == 0);
        // local entries are stored as byte offsets of the staged float4 slots (index << 4) while the most
        // populous neighbourhood, dummy slot included, stays below 4096 atoms
        int lshift = (ctx->nl_last_n == n && ctx->nl_last_max_pop > 4094) ? 0 : 4;
        bool use_staged = !ctx->pairs_staged_off;
        for (int attempt = 0;; ++attempt) {
            // the staging rows must fit the 227 KB a block can opt into (minus the kernel's static shared memory)
            const int cap_row_max = (int)(((size_t)232448 - 1024 - pairs_smem(0, local)) / (NL_WARPS * (local ? sizeof(uint16_t) : sizeof(uint32_t)))) & ~31;
            if (cap_row > cap_row_max)
                return cleanup(sqeq_fail(ctx, SQEQ_ECAPACITY,
                        "sqeq_nl_build: a row has %d neighbours; rows above %d are not supported", cap_row, cap_row_max));
            const size_t esize = local ? sizeof(uint16_t) : sizeof(uint32_t);
            if (!nl->nbr) NL_TRY(pool_alloc(ctx, (void**)&nl->nbr, esize * capacity));
            NLCounters init = {};
            for (int d = 0; d < 3; ++d) init.ex.L[d] = g.L[d];
            init.ex.rl2 = g.rl2;
            *hinit = init;
            NL_CUDA(cudaMemcpyAsync(ctr, hinit, sizeof(NLCounters), cudaMemcpyHostToDevice, st));
            // the staged sweep needs the neighbourhood size before the launch: a previous build of this system gives it
            // (+6 % and 64 atoms of room; a neighbourhood that outgrows it raises stage_overflow and k_pairs runs instead)
            int stage_cap = 0;
            if (local && use_staged && ctx->nl_last_n == n && ctx->nl_last_max_pop > 0) {
                stage_cap = (int)(1.06 * ctx->nl_last_max_pop) + 64;
                const size_t sm = sizeof(float4) * ((size_t)stage_cap + 33) + (size_t)NLS_WARPS * cap_row * sizeof(uint16_t);
                if (stage_cap > 65534 || sm > 110 * 1024) stage_cap = 0;      // two 512-thread blocks per SM
            }
            NL_TRY(launch_pairs(ctx, nl, pos, g, local, local ? lshift : 0, est_row, cap_row, capacity, ctr, st, stage_cap));
            NL_CUDA(cudaMemcpyAsync(h, ctr, sizeof(NLCounters), cudaMemcpyDeviceToHost, st));
            NL_CUDA(cudaMemcpyAsync(h_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, st));
            NL_CUDA(cudaStreamSynchronize(st));
            if (h_flag[0] & 1)
                return cleanup(sqeq_fail(ctx, SQEQ_EINVAL,
                                         "sqeq_nl_build: a position is non-finite or more than 127 box lengths away"));
            if (h->stage_overflow) { use_staged = false; if (attempt < 3) continue; }
            const bool row_ok = h->max_row <= cap_row, cap_ok = h->cursor <= capacity;
            const bool fmt_ok = !local || (h->max_pop <= 65534 && ((size_t)h->max_pop + 1) * sizeof(float4) <= REAL_STAGE_MAX_BYTES);
            const bool shift_ok = !local || !fmt_ok || lshift == 0 || h->max_pop <= 4094;
            if (row_ok && cap_ok && fmt_ok && shift_ok) break;
            if (attempt >= 3)
                return cleanup(sqeq_fail(ctx, SQEQ_ECAPACITY, "sqeq_nl_build: sizing did not converge"));
            if (!row_ok) cap_row = (h->max_row + 31) & ~31;
            if (!cap_ok || !fmt_ok) {
                NL_CUDA(cudaFreeAsync(nl->nbr, st));
                nl->nbr = nullptr;
                // the cursor of a failed pass is not reproducible (rows take their places in the order warps
                // finish, so which rows fall back to the global cursor varies): leave room for every group to
                // spill one padded row, plus 2 %
                if (!cap_ok) capacity = (size_t)h->cursor + (size_t)h->cursor / 50 +
                                        (size_t)nl->gg.ng[0] * nl->gg.ng[1] * nl->gg.ng[2] * (size_t)cap_row;
                if (!fmt_ok) local = false;
            }
            if (!shift_ok) lshift = 0;
        }
        nl->fmt = local ? 1 : 0;
        nl->max_pop = local ? h->max_pop : 0;
        nl->lshift = local ? lshift : 0;
        ctx->nl_last_max_pop = h->max_pop;
        ctx->nl_last_fmt = nl->fmt;
        nl->n_directed = (int64_t)h->pairs;
        nl->n_slots = (int64_t)h->cursor;
        nl->max_row = h->max_row;
        ctx->nl_last_n = n;
        ctx->nl_last_total = nl->n_slots;
        ctx->nl_last_pairs = nl->n_directed;
        ctx->nl_last_max_row = nl->max_row;
    }
    *out = nl;
    ctx->lists.push_back(nl);
    cleanup(SQEQ_OK);
    return SQEQ_OK;
#undef NL_TRY
#undef NL_CUDA
}

// Largest distance any atom has moved since the list was built (plain difference of caller positions: an atom
// that crossed the box is still the same unwrapped coordinate to the caller).  A list with cutoff rc + skin
// stays complete for r < rc while this is below skin/2 (cfg 4 recipe).
// vel != NULL: the displacement the atom will have after moving on by vel * dt (the position update of the next
// MD step, up to its dt^2 a/2 term)
__global__ void k_max_drift(int64_t n, const float* __restrict__ pos, const float* __restrict__ pos0,
                            const float* __restrict__ vel, float dt, unsigned* __restrict__ out)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    float d2 = 0.f;
    if (i < n) {
        float dx = pos[3 * i] - pos0[3 * i], dy = pos[3 * i + 1] - pos0[3 * i + 1], dz = pos[3 * i + 2] - pos0[3 * i + 2];
        if (vel) { dx = fmaf(dt, vel[3 * i], dx); dy = fmaf(dt, vel[3 * i + 1], dy); dz = fmaf(dt, vel[3 * i + 2], dz); }
        d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        if (!(d2 == d2)) d2 = __int_as_float(0x7f800000);      // NaN position: report +inf
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, o));
    if ((threadIdx.x & 31) == 0 && d2 > 0.f) atomicMax(out, __float_as_uint(d2));   // non-negative floats order as uints
}

// enqueue only: *d_out (device word, zeroed here) <- bits of the largest squared displacement
int nl_max_drift_enqueue(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* pos, const float* vel, double dt,
                         unsigned* d_out)
{
    cudaStream_t st = ctx->stream;
    CUDA_TRY(ctx, cudaMemsetAsync(d_out, 0, sizeof(unsigned), st));
    k_max_drift<<<ceil_div(nl->n, 256), 256, 0, st>>>(nl->n, pos, nl->pos0, vel, (float)dt, d_out);
    KERNEL_CHECK(ctx);
    return SQEQ_OK;
}

int nl_max_drift_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* pos, const float* vel, double dt,
                      double* max_drift)
{
    cudaStream_t st = ctx->stream;
    unsigned* d_out = (unsigned*)((double*)ctx->scal.p + 12);        // a scratch word of the scalar block
    CUDA_TRY(ctx, cudaMemsetAsync(d_out, 0, sizeof(unsigned), st));
    k_max_drift<<<ceil_div(nl->n, 256), 256, 0, st>>>(nl->n, pos, nl->pos0, vel, (float)dt, d_out);
    KERNEL_CHECK(ctx);
    unsigned* h = (unsigned*)(ctx->h_scal + 12);
    CUDA_TRY(ctx, cudaMemcpyAsync(h, d_out, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    float d2;
    memcpy(&d2, h, sizeof(float));
    *max_drift = sqrt((double)d2);
    return SQEQ_OK;
}

int nl_export_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, int32_t* oi, int32_t* oj, int8_t* shift3)
{
    cudaStream_t st = ctx->stream;
    const int64_t n = nl->n;
    if (nl->n_directed == 0) return SQEQ_OK;
    int* cnt = nullptr;
    int64_t* off = nullptr;
    int* flag = nullptr;
    uint32_t* expanded = nullptr;
    // temporaries from the context's stream-ordered pool, released on every path
    auto body = [&]() -> int {
        SQEQ_TRY(pool_alloc(ctx, (void**)&cnt, sizeof(int) * (n + 1)));
        SQEQ_TRY(pool_alloc(ctx, (void**)&off, sizeof(int64_t) * (n + 1)));
        SQEQ_TRY(pool_alloc(ctx, (void**)&flag, sizeof(int)));
        CUDA_TRY(ctx, cudaMemsetAsync(cnt, 0, sizeof(int) * (n + 1), st));
        CUDA_TRY(ctx, cudaMemsetAsync(flag, 0, sizeof(int), st));
        // a 16-bit local list is expanded to j | code entries first (same row offsets)
        const uint32_t* nbr32 = (const uint32_t*)nl->nbr;
        if (nl->fmt == 1) {
            SQEQ_TRY(pool_alloc(ctx, (void**)&expanded, sizeof(uint32_t) * (size_t)nl->n_slots));
            k_local_to_global<<<nl->gg.ng[0] * nl->gg.ng[1] * nl->gg.ng[2], 256, 0, st>>>(
                nl->cell_start, nl->gg, nl->row_start, nl->row_len, (const uint16_t*)nl->nbr, nl->lshift, expanded);
            KERNEL_CHECK(ctx);
            nbr32 = expanded;
        }
        k_export_count<<<ceil_div(n * 32, 256), 256, 0, st>>>(n, nl->row_start, nl->row_len, nbr32, nl->perm, cnt);
        KERNEL_CHECK(ctx);
        SQEQ_TRY(exclusive_scan<int>(ctx, n + 1, cnt, off, st));
        k_export_fill<<<(unsigned)n, 256, 0, st>>>(n, nl->row_start, nl->row_len, nbr32, nl->perm, nl->wrapc, off,
                                                    oi, oj, shift3, flag);
        KERNEL_CHECK(ctx);
        return SQEQ_OK;
    };
    const int r = body();
    int h_flag = 0;
    int64_t total = 0;
    if (r == SQEQ_OK) {
        cudaMemcpyAsync(&h_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
        cudaMemcpyAsync(&total, off + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    for (void* p : {(void*)cnt, (void*)off, (void*)flag, (void*)expanded})
        if (p) cudaFreeAsync(p, st);
    if (r != SQEQ_OK) return r;
    if (e != cudaSuccess) return sqeq_fail(ctx, SQEQ_ECUDA, "sqeq_nl_export: %s", cudaGetErrorString(e));
    if (h_flag & 2) return sqeq_fail(ctx, SQEQ_ECAPACITY, "sqeq_nl_export: a row has more than %d upper neighbours", EXPORT_CAP);
    if (total * 2 != nl->n_directed)
        return sqeq_fail(ctx, SQEQ_ECUDA, "sqeq_nl_export: list is not symmetric (%lld upper entries, %lld directed)",
                         (long long)total, (long long)nl->n_directed);
    return SQEQ_OK;
}

// mode 0: ELLPACK rows [n][K]; mode 1: directed COO of n_directed entries sorted by (i, j)
int nl_export_rows_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, int mode, int K, int32_t* oi, int32_t* oj, int8_t* shift3,
                        int32_t* counts)
{
    cudaStream_t st = ctx->stream;
    const int64_t n = nl->n;
    if (nl->max_row > EXPORT_ROW_CAP)
        return sqeq_fail(ctx, SQEQ_ECAPACITY, "neighbour export: a row has %d neighbours, more than %d", nl->max_row, EXPORT_ROW_CAP);
    uint32_t* expanded = nullptr;
    int* cnt = nullptr;
    int64_t* off = nullptr;
    auto body = [&]() -> int {
        const uint32_t* nbr32 = (const uint32_t*)nl->nbr;
        if (nl->fmt == 1 && nl->n_slots > 0) {
            SQEQ_TRY(pool_alloc(ctx, (void**)&expanded, sizeof(uint32_t) * (size_t)nl->n_slots));
            k_local_to_global<<<nl->gg.ng[0] * nl->gg.ng[1] * nl->gg.ng[2], 256, 0, st>>>(
                nl->cell_start, nl->gg, nl->row_start, nl->row_len, (const uint16_t*)nl->nbr, nl->lshift, expanded);
            KERNEL_CHECK(ctx);
            nbr32 = expanded;
        }
        if (mode == 1) {
            SQEQ_TRY(pool_alloc(ctx, (void**)&cnt, sizeof(int) * (n + 1)));
            SQEQ_TRY(pool_alloc(ctx, (void**)&off, sizeof(int64_t) * (n + 1)));
            CUDA_TRY(ctx, cudaMemsetAsync(cnt, 0, sizeof(int) * (n + 1), st));
            k_row_len_orig<<<ceil_div(n, 256), 256, 0, st>>>(n, nl->row_len, nl->perm, cnt);
            KERNEL_CHECK(ctx);
            SQEQ_TRY(exclusive_scan<int>(ctx, n + 1, cnt, off, st));
        }
        const size_t sm = sizeof(int) * 2 * EXPORT_ROW_CAP;
        CUDA_TRY(ctx, cudaFuncSetAttribute(k_export_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        k_export_rows<<<(unsigned)n, 256, sm, st>>>(nl->row_start, nl->row_len, nbr32, nl->perm, nl->wrapc, K, off,
                                                     mode == 1 ? oi : nullptr, oj, shift3, counts);
        KERNEL_CHECK(ctx);
        return SQEQ_OK;
    };
    const int r = body();
    cudaError_t e = cudaStreamSynchronize(st);
    for (void* p : {(void*)expanded, (void*)cnt, (void*)off})
        if (p) cudaFreeAsync(p, st);
    if (r != SQEQ_OK) return r;
    if (e != cudaSuccess) return sqeq_fail(ctx, SQEQ_ECUDA, "neighbour export: %s", cudaGetErrorString(e));
    return SQEQ_OK;
}
