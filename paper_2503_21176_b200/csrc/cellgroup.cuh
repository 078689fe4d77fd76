// cellgroup.cuh -- the NEIGHBOURHOOD of a group of neighbour-list cells, shared by the pair
// enumeration (nlist.cu) and the shared-memory-staged real-space kernel (realspace.cu).
//
// Cells are z-fastest in memory, so the cells a group of g0 x g1 x g2 cells can interact with --
// the group widened by the stencil half-width w on every side -- are (g0+2w)(g1+2w) COLUMNS, each
// column at most three contiguous runs of atoms (one per periodic image along z): the PIECES.
// Concatenating the pieces in (column, image) order gives every atom of the neighbourhood, image
// by image, a LOCAL index.  Both kernels derive the same layout from cell_start, so a neighbour
// list can store 16-bit local indices and the real-space kernel can stage the neighbourhood in
// shared memory -- with the image shift already applied -- and gather from there.
#pragma once
#include <stdint.h>

#define GRP_G 2                      // cells per group and axis
#define GRP_MAXCOL 36                // (GRP_G + 2*2)^2
#define GRP_MAXPIECE (3 * GRP_MAXCOL)

struct GroupGeom {
    int nc[3];     // cells per axis
    int ng[3];     // groups per axis
    int w[3];      // stencil half-width per axis (1 or 2)
};

struct GroupPiece {
    int gbeg;      // first sorted-atom index of the run
    int len;       // atoms in the run (0: piece absent)
    int lbase;     // local index of its first atom
    int code;      // image code (sx+1)*9 + (sy+1)*3 + (sz+1) of the run relative to the group
};

struct GroupInfo {
    int c0[3];     // first cell of the group
    int ge[3];     // cells of the group per axis (< GRP_G at the upper box faces)
    int ncoly;     // columns along y: ge[1] + 2 w[1]
    int ncol;      // columns
    int pop;       // atoms in the neighbourhood (all images)
};

// u in [-nc, 2nc) -> wrapped cell index and image shift; false if |shift| would exceed 1
__device__ __forceinline__ bool grp_wrap(int& u, int nc, int& sh)
{
    sh = 0;
    if (u < 0) { u += nc; sh = -1; } else if (u >= nc) { u -= nc; sh = 1; }
    return u >= 0 && u < nc;
}

// Block-cooperative (>= 128 threads, all threads must call): pieces[col*3 + p], p = image along z + 1.
// `scratch` is one int of shared memory.
__device__ __forceinline__ GroupInfo group_layout(const GroupGeom& gg, const int* __restrict__ cell_start,
                                                  int group_id, GroupPiece* pieces, int* scratch)
{
    GroupInfo gi;
    int b = group_id;
    const int bz = b % gg.ng[2]; b /= gg.ng[2];
    const int by = b % gg.ng[1];
    const int bx = b / gg.ng[1];
    gi.c0[0] = bx * GRP_G; gi.c0[1] = by * GRP_G; gi.c0[2] = bz * GRP_G;
#pragma unroll
    for (int d = 0; d < 3; ++d) gi.ge[d] = min(GRP_G, gg.nc[d] - gi.c0[d]);
    gi.ncoly = gi.ge[1] + 2 * gg.w[1];
    gi.ncol = (gi.ge[0] + 2 * gg.w[0]) * gi.ncoly;
    const int np = gi.ncol * 3;
    const int tid = threadIdx.x;
    int len = 0;
    if (tid < np) {
        const int col = tid / 3, p = tid - col * 3;
        int ux = gi.c0[0] - gg.w[0] + col / gi.ncoly, uy = gi.c0[1] - gg.w[1] + col % gi.ncoly, shx, shy;
        bool valid = grp_wrap(ux, gg.nc[0], shx);
        valid = grp_wrap(uy, gg.nc[1], shy) && valid;
        const int ncz = gg.nc[2], shz = p - 1;
        const int zlo = max(gi.c0[2] - gg.w[2], shz * ncz), zhi = min(gi.c0[2] + gi.ge[2] - 1 + gg.w[2], (shz + 1) * ncz - 1);
        GroupPiece pc;
        pc.gbeg = 0; pc.len = 0; pc.lbase = 0;
        pc.code = (shx + 1) * 9 + (shy + 1) * 3 + (shz + 1);
        if (valid && zhi >= zlo) {
            const int colw = (ux * gg.nc[1] + uy) * ncz - shz * ncz;
            pc.gbeg = cell_start[colw + zlo];
            pc.len = cell_start[colw + zhi + 1] - pc.gbeg;
        }
        len = pc.len;
        pieces[tid] = pc;
    }
    // exclusive scan of the piece lengths over the first 128 threads (4 warps)
    __shared__ int grp_wsum[4];
    const int lane = tid & 31, wid = tid >> 5;
    int incl = len;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    if (wid < 4 && lane == 31) grp_wsum[wid] = incl;
    __syncthreads();
    if (tid < np) {
        int off = 0;
        for (int k = 0; k < wid; ++k) off += grp_wsum[k];
        pieces[tid].lbase = off + incl - len;
    }
    if (tid == 0) *scratch = grp_wsum[0] + grp_wsum[1] + grp_wsum[2] + grp_wsum[3];
    __syncthreads();
    gi.pop = *scratch;
    return gi;
}
