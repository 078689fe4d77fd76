// pme.cu -- smooth Particle Mesh Ewald, Alg. 2, steps a-4 ... a-8:
//   spread (order-p cardinal B-splines) -> cuFFT R2C -> influence multiply (+ E_rec) -> cuFFT C2R
//   -> gather of phi_rec and F_rec.  Conventions are DESIGN.md R-PME: weight M_p(w+j) on grid index
//   f-j, unnormalised transforms (no 1/K^3), G(m) = B(m) exp(-pi^2 mt^2/alpha^2)/(pi V mt^2), G(0)=0.
// cuFFT does the two 3-D transforms (north_star allows it; timed as separate stages).
#include <math.h>
#include <stdlib.h>

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
// a-4, Alg. 2 step 1.  A block takes SPREAD_APB consecutive atoms: 3 threads per
// atom evaluate the per-axis weights into shared memory, then the block sweeps the atoms' P^2 (x,y)
// ROWS, one row of P z-contiguous points per thread (flat row index -> every lane busy, index
// arithmetic paid once per row instead of once per point).  A row is added to the grid with
// 8-byte vector reductions (red.global.add.v2.f32) on even-aligned pairs; K2 is even, so a pair
// never straddles the periodic boundary, and an odd row start is padded with a zero on each side.
#define SPREAD_APB 64
__device__ __forceinline__ void red_add_v2(float* addr, float a, float b)
{
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}

template <int P>
__global__ void __launch_bounds__(256)
k_spread(int64_t n, const float4* __restrict__ frac, const int4* __restrict__ base, int K0, int K1, int K2,
         float* __restrict__ grid)
{
    __shared__ float wt[SPREAD_APB][3][P];
    __shared__ int4 sb[SPREAD_APB];
    const int64_t s0 = blockIdx.x * (int64_t)SPREAD_APB;
    const int na = (int)min((int64_t)SPREAD_APB, n - s0);
    if (threadIdx.x < 3 * SPREAD_APB) {
        const int at = threadIdx.x / 3, ax = threadIdx.x % 3;
        if (at < na) {
            const float4 fw = frac[s0 + at];
            float th[P], dth[P];
            bspline_weights<P>(ax == 0 ? fw.x : (ax == 1 ? fw.y : fw.z), th, dth);
#pragma unroll
            for (int j = 0; j < P; ++j) wt[at][ax][j] = th[j];
            if (ax == 0) {
                int4 f = base[s0 + at];
                f.w = __float_as_int(fw.w);
                sb[at] = f;
            }
        }
    }
    __syncthreads();
    const int rows = na * P * P;
    for (int R = threadIdx.x; R < rows; R += blockDim.x) {
        const int at = R / (P * P), row = R % (P * P);
        const int a = row / P, b = row % P;
        const int4 f = sb[at];
        const float w2 = __int_as_float(f.w) * wt[at][0][a] * wt[at][1][b];
        if (w2 == 0.f) continue;
        int gx = f.x - a; gx += gx < 0 ? K0 : 0;
        int gy = f.y - b; gy += gy < 0 ? K1 : 0;
        float* rowp = grid + ((size_t)gx * K1 + gy) * K2;
        // ascending z: point i (0..P-1) is grid index zs+i and carries theta_z[P-1-i]
        int zs = f.z - (P - 1); zs += zs < 0 ? K2 : 0;
        const int odd = zs & 1;
        float ext[P + 2];
        ext[0] = 0.f; ext[P + 1] = 0.f;
#pragma unroll
        for (int i = 0; i < P; ++i) ext[i + 1] = w2 * wt[at][2][P - 1 - i];
        int pz = zs - odd;                       // even start of the first pair
#pragma unroll
        for (int j = 0; j <= P / 2; ++j) {
            if (j == P / 2 && !odd && !(P & 1)) break;      // odd P: (P + 1)/2 pairs either way, one zero pad
            const float lo = odd ? ext[2 * j] : ext[2 * j + 1];
            const float hi = odd ? ext[2 * j + 1] : ext[2 * j + 2];
            red_add_v2(rowp + pz, lo, hi);
            pz += 2; pz -= pz >= K2 ? K2 : 0;
        }
    }
}

// -------------------------------------------------------------------------------------- influence
// a-6, Alg. 2 step 3: Qhat(m) *= G(m); E_rec = 1/2 sum_m G |Qhat|^2 with Hermitian
// weights on the half spectrum.  G is formed in fp64 from three per-axis tables.
__global__ void __launch_bounds__(256)
k_influence(int K0, int K1, int K2h, int K2, const float* __restrict__ tab, float inv_piV,
            float2* __restrict__ spec, double* __restrict__ e_out)
{
    // per-axis fp32 tables (built in fp64 on the host): Bg_d[m] = |b_d(m)|^2 exp(-pi^2 mt_d^2/alpha^2), s_d[m] = mt_d^2
    const int total_rows = K0 * K1;
    const float* Bg0 = tab;       const float* s0 = Bg0 + K0;
    const float* Bg1 = s0 + K0;   const float* s1 = Bg1 + K1;
    const float* Bg2 = s1 + K1;   const float* s2 = Bg2 + K2;
    double e = 0.0;
    // one warp per (m0, m1) row, lanes along m2 (coalesced; no per-element division by K2h)
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
    for (int row = warp; row < total_rows; row += nwarp) {
        const int m0 = row / K1, m1 = row - m0 * K1;
        const float bg01 = Bg0[m0] * Bg1[m1] * inv_piV, s01 = s0[m0] + s1[m1];
        float2* srow = spec + (size_t)row * K2h;
        float er = 0.f;
        for (int m2 = lane; m2 < K2h; m2 += 32) {
            float G = 0.f;
            if (row | m2) G = __fdividef(bg01 * Bg2[m2], s01 + s2[m2]);
            float2 z = srow[m2];
            const float w = (m2 == 0 || 2 * m2 == K2) ? 0.5f : 1.0f;     // 1/2 * (1 or 2)
            er = fmaf(w * G, fmaf(z.x, z.x, z.y * z.y), er);
            z.x *= G;
            z.y *= G;
            srow[m2] = z;
        }
        e += (double)er;
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

// -------------------------------------------------------------------------------------- fused x-axis pass
// north_star: "the influence-function convolution fused into the FFT pre- and post-passes".  The 3-D transforms
// are split as  [cuFFT 2-D R2C over (y,z), batched over x]  ->  THIS KERNEL  ->  [cuFFT 2-D C2R, batched over x]:
// for a tile of XF_TJ neighbouring (m1, m2) lines the block holds the whole x-extent in shared memory, runs the
// forward 1-D transform along x (Stockham autosort, radices 2/3/4/5), multiplies by G(m) and accumulates
// E_rec = 1/2 sum w G |Qhat|^2, runs the inverse transform along x and writes the lines back: the spectrum is read
// and written ONCE where cuFFT's two x-passes and a separate influence kernel touched it three times.
#define XF_TJ 16
#define XF_NT 320
#define XF_MAXPASS 12
struct XfPlan {
    int N;                      // K0
    int npass;
    int radix[XF_MAXPASS];
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// one Stockham pass of radix R over all XF_TJ lines: in[x][tj] -> out[x][tj].  INV: conjugate twiddles.
template <int R, bool INV>
__device__ __forceinline__ void xf_pass(const float2* __restrict__ in, float2* __restrict__ out, const float2* __restrict__ W,
                                        int N, int Ns)
{
    const int nb = N / R;                                   // butterflies per line
    const int tstep = N / (Ns * R);                         // twiddle index step: angle = -2 pi t k / (Ns R)
    const float inv_ns = 1.f / (float)Ns;
    for (int task = threadIdx.x; task < nb * XF_TJ; task += XF_NT) {
        const int j = task / XF_TJ, tj = task - j * XF_TJ;
        const int jq = __float2int_rd(((float)j + 0.5f) * inv_ns);     // j / Ns, exact for j < 2^20
        const int k = j - jq * Ns;
        float2 v[R];
#pragma unroll
        for (int t = 0; t < R; ++t) {
            v[t] = in[(j + t * nb) * XF_TJ + tj];
            if (t > 0) {
                float2 w = W[t * k * tstep];                   // t k < R Ns, so the index stays below N
                if (INV) w.y = -w.y;
                v[t] = cmul(v[t], w);
            }
        }
        const float sg = INV ? 1.f : -1.f;                  // forward: e^{-i...}
        if (R == 2) {
            const float2 a = v[0], b = v[1];
            v[0] = make_float2(a.x + b.x, a.y + b.y);
            v[1] = make_float2(a.x - b.x, a.y - b.y);
        } else if (R == 4) {
            const float2 a = make_float2(v[0].x + v[2].x, v[0].y + v[2].y), b = make_float2(v[0].x - v[2].x, v[0].y - v[2].y);
            const float2 c = make_float2(v[1].x + v[3].x, v[1].y + v[3].y), d = make_float2(v[1].x - v[3].x, v[1].y - v[3].y);
            const float2 id = make_float2(-sg * d.y, sg * d.x);   // (sg i) d : forward -i d
            v[0] = make_float2(a.x + c.x, a.y + c.y);
            v[2] = make_float2(a.x - c.x, a.y - c.y);
            v[1] = make_float2(b.x + id.x, b.y + id.y);
            v[3] = make_float2(b.x - id.x, b.y - id.y);
        } else if (R == 3) {
            const float c3 = -0.5f, s3 = sg * 0.86602540378443865f;
            const float2 s = make_float2(v[1].x + v[2].x, v[1].y + v[2].y), d = make_float2(v[1].x - v[2].x, v[1].y - v[2].y);
            const float2 m = make_float2(v[0].x + c3 * s.x, v[0].y + c3 * s.y);
            const float2 id = make_float2(-s3 * d.y, s3 * d.x);   // i s3 d
            v[0] = make_float2(v[0].x + s.x, v[0].y + s.y);
            v[1] = make_float2(m.x + id.x, m.y + id.y);
            v[2] = make_float2(m.x - id.x, m.y - id.y);
        } else if (R == 5) {
            const float c1 = 0.30901699437494742f, c2 = -0.80901699437494742f;
            const float s1 = sg * 0.95105651629515357f, s2 = sg * 0.58778525229247313f;
            const float2 a1 = make_float2(v[1].x + v[4].x, v[1].y + v[4].y), b1 = make_float2(v[1].x - v[4].x, v[1].y - v[4].y);
            const float2 a2 = make_float2(v[2].x + v[3].x, v[2].y + v[3].y), b2 = make_float2(v[2].x - v[3].x, v[2].y - v[3].y);
            const float2 m1 = make_float2(v[0].x + c1 * a1.x + c2 * a2.x, v[0].y + c1 * a1.y + c2 * a2.y);
            const float2 m2 = make_float2(v[0].x + c2 * a1.x + c1 * a2.x, v[0].y + c2 * a1.y + c1 * a2.y);
            const float2 n1 = make_float2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
            const float2 n2 = make_float2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
            v[0] = make_float2(v[0].x + a1.x + a2.x, v[0].y + a1.y + a2.y);
            v[1] = make_float2(m1.x - n1.y, m1.y + n1.x);          // m1 + i n1
            v[4] = make_float2(m1.x + n1.y, m1.y - n1.x);
            v[2] = make_float2(m2.x - n2.y, m2.y + n2.x);
            v[3] = make_float2(m2.x + n2.y, m2.y - n2.x);
        }
        const int j0 = jq * Ns * R + k;
#pragma unroll
        for (int t = 0; t < R; ++t) out[(j0 + t * Ns) * XF_TJ + tj] = v[t];
    }
}

template <bool INV>
__device__ __forceinline__ float2* xf_transform(float2* a, float2* b, const float2* W, const XfPlan& pl)
{
    int Ns = 1;
    for (int p = 0; p < pl.npass; ++p) {
        const int R = pl.radix[p];
        if (R == 4) xf_pass<4, INV>(a, b, W, pl.N, Ns);
        else if (R == 2) xf_pass<2, INV>(a, b, W, pl.N, Ns);
        else if (R == 3) xf_pass<3, INV>(a, b, W, pl.N, Ns);
        else xf_pass<5, INV>(a, b, W, pl.N, Ns);
        Ns *= R;
        __syncthreads();
        float2* t = a; a = b; b = t;
    }
    return a;                                               // where the result is
}

__global__ void __launch_bounds__(XF_NT)
k_xline_influence(XfPlan pl, int K1, int K2h, int K2, const float* __restrict__ tab, float inv_piV,
                  const float2* __restrict__ Wg, float2* __restrict__ spec, double* __restrict__ e_out)
{
    extern __shared__ __align__(16) float2 xf_sh[];         // W[N] | buf A [N][TJ] | buf B [N][TJ]
    const int N = pl.N;
    float2* W = xf_sh;
    float2* A = W + N;
    float2* B = A + N * XF_TJ;
    const int nline = K1 * K2h;
    const int j0 = blockIdx.x * XF_TJ;
    for (int i = threadIdx.x; i < N; i += XF_NT) W[i] = Wg[i];
    for (int e = threadIdx.x; e < N * XF_TJ; e += XF_NT) {
        const int x = e / XF_TJ, tj = e - x * XF_TJ;
        A[e] = j0 + tj < nline ? spec[(size_t)x * nline + j0 + tj] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    float2* F = xf_transform<false>(A, B, W, pl);
    float2* O = F == A ? B : A;
    // influence multiply (Alg. 2 step 3) and the energy, as in k_influence
    const float* Bg0 = tab;       const float* s0 = Bg0 + N;
    const float* Bg1 = s0 + N;    const float* s1 = Bg1 + K1;
    const float* Bg2 = s1 + K1;   const float* s2 = Bg2 + K2;
    float er = 0.f;
    static_assert(XF_NT % XF_TJ == 0, "a thread keeps its line");
    // a thread always meets the same line tj (XF_NT is a multiple of XF_TJ): its (m1, m2) factors once
    const int tj_ = threadIdx.x % XF_TJ, jl = j0 + tj_;
    const bool line_on = jl < nline;
    const int m1 = line_on ? jl / K2h : 0, m2 = line_on ? jl - m1 * K2h : 0;
    const float bg12 = Bg1[m1] * Bg2[m2] * inv_piV, s12 = s1[m1] + s2[m2];
    const float w = !line_on ? 0.f : ((m2 == 0 || 2 * m2 == K2) ? 0.5f : 1.0f);
    for (int e = threadIdx.x; e < N * XF_TJ; e += XF_NT) {
        const int m0 = e / XF_TJ;
        float G = 0.f;
        if (line_on && (m0 | jl)) G = __fdividef(Bg0[m0] * bg12, s0[m0] + s12);
        float2 z = F[e];
        er = fmaf(w * G, fmaf(z.x, z.x, z.y * z.y), er);
        z.x *= G; z.y *= G;
        F[e] = z;
    }
    __syncthreads();
    float2* R = xf_transform<true>(F, O, W, pl);
    for (int e = threadIdx.x; e < N * XF_TJ; e += XF_NT) {
        const int x = e / XF_TJ, tj = e - x * XF_TJ;
        if (j0 + tj < nline) spec[(size_t)x * nline + j0 + tj] = R[e];
    }
    if (e_out) {
        double e = (double)er;
        __shared__ double red[XF_NT / 32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int k = 0; k < XF_NT / 32; ++k) t += red[k];
            atomicAdd(e_out, t);
        }
    }
}

// -------------------------------------------------------------------------------------- gather
// a-8, Alg. 2 step 5: phi_i = sum W Phi;  F_i,x = -q_i (K_x/L_x) sum dW_x Phi.
// One warp per atom, one (x,y) ROW of P z-contiguous points per lane: per row the z sums
// s0 = sum_c theta_z Phi and s1 = sum_c dtheta_z Phi cost 2 FMAs per point, and the x,y factors are
// applied once per row.  For P = 6 the 4 rows beyond the first 32 are handed out point by point to
// lanes 0..23 so that no pass runs with 4 active lanes.
template <int P, bool FORCE>
__device__ __forceinline__ void gather_row(const float* __restrict__ grid, const float (*w)[P], int a, int b,
                                           int c0, int c1, const int4 f, int K0, int K1, int K2,
                                           float& ph, float& gx_, float& gy_, float& gz_)
{
    int gx = f.x - a; gx += gx < 0 ? K0 : 0;
    int gy = f.y - b; gy += gy < 0 ? K1 : 0;
    const float* rowp = grid + ((size_t)gx * K1 + gy) * K2;
    float s0 = 0.f, s1 = 0.f;
#pragma unroll
    for (int c = 0; c < P; ++c) {
        if (c < c0 || c >= c1) continue;
        int gz = f.z - c; gz += gz < 0 ? K2 : 0;
        const float v = __ldg(rowp + gz);
        s0 = fmaf(w[2][c], v, s0);
        if (FORCE) s1 = fmaf(w[5][c], v, s1);
    }
    const float tx = w[0][a], ty = w[1][b];
    ph = fmaf(tx * ty, s0, ph);
    if (FORCE) {
        gx_ = fmaf(w[3][a] * ty, s0, gx_);
        gy_ = fmaf(tx * w[4][b], s0, gy_);
        gz_ = fmaf(tx * ty, s1, gz_);
    }
}

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
    const float (*w)[P] = wt[wid];
    float ph = 0.f, gx_ = 0.f, gy_ = 0.f, gz_ = 0.f;
    if (P == 6) {
        gather_row<P, FORCE>(grid, w, lane / P, lane % P, 0, P, f, K0, K1, K2, ph, gx_, gy_, gz_);
        if (lane < 24) {                       // rows 32..35 = (a = 5, b = 2..5), one point per lane
            const int c = lane % P;
            gather_row<P, FORCE>(grid, w, 5, 2 + lane / P, c, c + 1, f, K0, K1, K2, ph, gx_, gy_, gz_);
        }
    } else {
        for (int row = lane; row < P * P; row += 32)
            gather_row<P, FORCE>(grid, w, row / P, row % P, 0, P, f, K0, K1, K2, ph, gx_, gy_, gz_);
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

// -------------------------------------------------------------------------------------- tiles
// Shared-memory tiles for spread and gather.  The atoms arrive in the neighbour list's cell-major
// order (cells z-fastest), so a GROUP of g0 x g1 x g2 cells is g0*g1 contiguous atom runs that sit
// in one compact region of the grid.  A block takes one group: its tile is the grid window
//   [o_d, o_d + T_d),  o_d = floor(c0_d K_d / nc_d) - M - (P-1),  T_d = floor(g_d K_d / nc_d) + 2 + 2M + (P-1)
// i.e. every point an atom of the group can touch while it has drifted less than M grid spacings
// since the list was built.  Spread accumulates into the tile (shared-memory atomics) and flushes
// it once with coalesced reductions; gather loads the tile once with coalesced loads and
// interpolates out of shared memory.  An atom whose footprint is not inside the window (it drifted
// further) takes the global-memory path inside the same kernel, so the result never depends on
// the drift bound.  Tile strides are padded on the host so that the 32 (x,y) rows a warp touches
// at once fall into distinct banks.  Atoms are processed in chunks of NT/4: three threads
// per atom evaluate its spline weights into a shared record (all lanes busy), then the rows follow.
struct TileGeom {
    int K[3];
    int nc[3];     // neighbour-list cells per axis
    int g[3];      // cells per group
    int ng[3];     // groups per axis
    int T[3];      // tile extent in grid points
    int ZS, XS;    // shared-memory strides: element (tx,ty,tz) at tx*XS + ty*ZS + tz
    int M;         // drift margin in grid points
    unsigned T1_magic;   // ceil(2^32 / T[1]): r / T[1] = umulhi(r, T1_magic) for r < 2^16
    unsigned nvz_magic;  // ceil(2^32 / (T[2]/4)): i / (T[2]/4) = umulhi(i, nvz_magic) for i < T[0] T[1] T[2]/4
};
#define TILE_MAXRANGES 16
#ifndef PME_ATOM_NT
#define PME_ATOM_NT 384       // threads per block of the one-thread-per-atom tile kernels
#endif
#define TILE_CHUNK(NT) ((NT) / 4)
// per-atom record (floats): theta_z[8] | dtheta_z[8] | theta_x[P] | theta_y[P] | dtheta_x[P] | dtheta_y[P]
#define REC_Z 0
#define REC_DZ 8
#define REC_X 16
#define REC_LEN(P) (16 + 4 * (P))

struct TileBlock {
    int o[3];          // tile origin (grid index of element 0; may be negative)
    int natoms;        // atoms of this group
};

// a in (-K, 2K) -> [0, K)
__device__ __forceinline__ int wrap1(int a, int K) { a += a < 0 ? K : 0; a -= a >= K ? K : 0; return a; }

// ranges of sorted-atom indices of the block's group; rpre = exclusive prefix of their lengths
__device__ __forceinline__ TileBlock tile_block_setup(const TileGeom& tg, const int* __restrict__ cell_start,
                                                       int P, int* rbeg, int* rpre)
{
    TileBlock tb;
    int b = blockIdx.x;
    const int bz = b % tg.ng[2]; b /= tg.ng[2];
    const int by = b % tg.ng[1];
    const int bx = b / tg.ng[1];
    const int c0[3] = {bx * tg.g[0], by * tg.g[1], bz * tg.g[2]};
    int gc[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        gc[d] = min(tg.g[d], tg.nc[d] - c0[d]);
        tb.o[d] = (int)((unsigned)(c0[d] * tg.K[d]) / (unsigned)tg.nc[d]) - tg.M - (P - 1);    // c0, K < 2^10
    }
    tb.o[2] &= ~3;      // z origin on a float4 boundary (K2 % 4 == 0): the window moves as 16-byte vectors
    const int nr = gc[0] * gc[1];
    if (threadIdx.x < nr) {
        const int cx = c0[0] + threadIdx.x / gc[1], cy = c0[1] + threadIdx.x % gc[1];
        const int col = (cx * tg.nc[1] + cy) * tg.nc[2] + c0[2];
        const int beg = cell_start[col];
        rbeg[threadIdx.x] = beg;
        rpre[threadIdx.x + 1] = cell_start[col + gc[2]] - beg;     // length, scanned below
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int acc = 0;
        rpre[0] = 0;
        for (int r = 0; r < nr; ++r) { acc += rpre[r + 1]; rpre[r + 1] = acc; }
        for (int r = nr; r < TILE_MAXRANGES; ++r) rpre[r + 1] = acc;
    }
    __syncthreads();
    tb.natoms = rpre[TILE_MAXRANGES];
    return tb;
}

__device__ __forceinline__ int tile_atom(int i, const int* rbeg, const int* rpre)
{
    int r = 0;
#pragma unroll
    for (int k = 1; k < TILE_MAXRANGES; ++k) r += (i >= rpre[k]);
    return rbeg[r] + (i - rpre[r]);
}

// Chunk setup by threads 0 .. 3*TILE_CHUNK(NT)-1 (thread = atom*3 + axis): spline weights into the atom's
// record, and by the axis-0 thread the atom's sorted index, raw base index + charge bits, and the
// linear tile offset of its base point (-1: footprint not inside the window).
// QSCALE (spread): theta_x is stored multiplied by q_i * qscale, so that a row's weight is one product.
template <int P, int NT, bool DERIV, bool QSCALE = false>
__device__ __forceinline__ void tile_chunk_setup(int ch, int na, const TileBlock& tb, const TileGeom& tg,
                                                 const float4* __restrict__ frac, const int4* __restrict__ base,
                                                 const int* rbeg, const int* rpre, float* rec, int4* sb,
                                                 int* stoff, int* sidx, float qscale = 1.f)
{
    if (threadIdx.x >= 3 * TILE_CHUNK(NT)) return;
    const int at = threadIdx.x / 3, ax = threadIdx.x % 3;
    if (at >= na) return;
    const int s = tile_atom(ch + at, rbeg, rpre);
    const float4 fw = frac[s];
    float th[P], dth[P];
    bspline_weights<P>(ax == 0 ? fw.x : (ax == 1 ? fw.y : fw.z), th, dth);
    float* r = rec + at * REC_LEN(P);
    const int o_t = ax == 2 ? REC_Z : REC_X + ax * P;
    const int o_d = ax == 2 ? REC_DZ : REC_X + (2 + ax) * P;
    const float ts = (QSCALE && ax == 0) ? fw.w * qscale : 1.f;
#pragma unroll
    for (int j = 0; j < P; ++j) {
        r[o_t + j] = QSCALE ? th[j] * ts : th[j];
        if (DERIV) r[o_d + j] = dth[j];
    }
    if (ax == 0) {
        int4 f = base[s];
        const int tx = wrap1(f.x - tb.o[0], tg.K[0]), ty = wrap1(f.y - tb.o[1], tg.K[1]),
                  tz = wrap1(f.z - tb.o[2], tg.K[2]);
        const bool in = tx >= P - 1 && tx < tg.T[0] && ty >= P - 1 && ty < tg.T[1] && tz >= P - 1 && tz < tg.T[2];
        stoff[at] = in ? tx * tg.XS + ty * tg.ZS + tz : -1;
        sidx[at] = s;
        f.w = __float_as_int(fw.w);
        sb[at] = f;
    }
}

// Moves the window between the grid and the tile as float4 vectors.  The z origin and K2 are multiples
// of 4, so a vector never straddles the periodic boundary; the tile side stays scalar (its row stride is
// odd).
// FLUSH: tile -> grid with red.global.add.v4.f32, all-zero vectors skipped; else grid -> tile.
__device__ __forceinline__ void red_add_v4(float* addr, float4 v)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

template <bool FLUSH, bool FIXED = false>
__device__ __forceinline__ void tile_move(float* tile, float* grid, const TileBlock& tb, const TileGeom& tg,
                                          float inv_scale = 1.f)
{
    // flat index over the window's float4 vectors (z fastest): consecutive threads take consecutive vectors
    // of a row, TILE_MOVE_U vectors per thread are in flight at once (loads first, then the shared stores)
    constexpr int U = 4;
    const int K0 = tg.K[0], K1 = tg.K[1], K2 = tg.K[2];
    const int nvz = tg.T[2] >> 2;
    const int nvec = tg.T[0] * tg.T[1] * nvz;
    for (int i0 = threadIdx.x; i0 < nvec; i0 += blockDim.x * U) {
        float4 v[U];
        float* tp[U];
        float* gp[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = min(i0 + u * (int)blockDim.x, nvec - 1);        // clamped: the store is predicated below
            const int r = (int)__umulhi((unsigned)i, tg.nvz_magic), tz = (i - r * nvz) << 2;
            const int tx = (int)__umulhi((unsigned)r, tg.T1_magic), ty = r - tx * tg.T[1];
            const int gx = wrap1(tb.o[0] + tx, K0), gy = wrap1(tb.o[1] + ty, K1), gz = wrap1(tb.o[2] + tz, K2);
            tp[u] = tile + tx * tg.XS + ty * tg.ZS + tz;
            gp[u] = grid + ((size_t)(gx * K1 + gy) * K2 + gz);
            if (!FLUSH) v[u] = __ldg((const float4*)gp[u]);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (i0 + u * (int)blockDim.x >= nvec) break;
            float* t = tp[u];
            if (FLUSH) {
                float4 w;
                if (FIXED) {
                    const int* it = (const int*)t;
                    w = make_float4(inv_scale * (float)it[0], inv_scale * (float)it[1], inv_scale * (float)it[2],
                                    inv_scale * (float)it[3]);
                } else {
                    w = make_float4(t[0], t[1], t[2], t[3]);
                }
                if (w.x != 0.f || w.y != 0.f || w.z != 0.f || w.w != 0.f) red_add_v4(gp[u], w);
            } else {
                t[0] = v[u].x; t[1] = v[u].y; t[2] = v[u].z; t[3] = v[u].w;
            }
        }
    }
}

// FIXED: the tile accumulates 32-bit fixed point with the native shared integer atomic (one ATOMS.ADD
// instead of a 7-instruction fp32 compare-and-swap loop that retries under contention).  The scale is
// per block: |tile point| <= sum_i |q_i| theta_x theta_y theta_z <= (2/3)^3 sum_i |q_i| over the block's
// atoms (2/3 = max of M_4, the largest cardinal B-spline peak of the supported orders), so
// S = 2^30 / ((2/3)^3 sum|q|) cannot overflow; one addition rounds by <= 0.5/S.
template <int P, int NT, bool FIXED>
__global__ void __launch_bounds__(NT)
k_spread_tile(const float4* __restrict__ frac, const int4* __restrict__ base,
              const int* __restrict__ cell_start, TileGeom tg, float* __restrict__ grid)
{
    extern __shared__ __align__(16) float tile[];
    __shared__ __align__(16) float rec[TILE_CHUNK(NT) * REC_LEN(P)];
    __shared__ int4 sb[TILE_CHUNK(NT)];
    __shared__ int stoff[TILE_CHUNK(NT)], sidx[TILE_CHUNK(NT)];
    __shared__ int rbeg[TILE_MAXRANGES], rpre[TILE_MAXRANGES + 1];
    const TileBlock tb = tile_block_setup(tg, cell_start, P, rbeg, rpre);
    if (tb.natoms == 0) return;
    const int K0 = tg.K[0], K1 = tg.K[1], K2 = tg.K[2];
    const int tsize = tg.XS * tg.T[0];
    for (int e = threadIdx.x; e < (tsize >> 2); e += blockDim.x) ((float4*)tile)[e] = make_float4(0.f, 0.f, 0.f, 0.f);   // 0.f and 0 share a bit pattern
    if (threadIdx.x < (tsize & 3)) tile[(tsize & ~3) + threadIdx.x] = 0.f;
    float scale = 1.f;
    if (FIXED) {
        __shared__ float s_part[NT / 32];
        float aq = 0.f;
        for (int i = threadIdx.x; i < tb.natoms; i += NT) aq += fabsf(frac[tile_atom(i, rbeg, rpre)].w);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) aq += __shfl_xor_sync(0xffffffffu, aq, o);
        if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = aq;
        __syncthreads();
        aq = 0.f;
#pragma unroll
        for (int k = 0; k < NT / 32; ++k) aq += s_part[k];
        scale = aq > 0.f ? 1073741824.f / (0.2962963f * aq * 1.0001f) : 1.f;
    }

    // thread <-> (atom slot, (x,y) row): the row (a, b) of a thread is fixed, NT / P^2 atoms are in flight per
    // pass, and the index arithmetic of a row is paid once per kernel instead of once per row
    constexpr int PP = P * P, APP = NT / PP;
    const int slot = threadIdx.x / PP, row = threadIdx.x - slot * PP;
    const int a = row / P, b = row - a * P;
    const int off_ab = a * tg.XS + b * tg.ZS;
    const float inv_scale = 1.f / scale;
    for (int ch = 0; ch < tb.natoms; ch += TILE_CHUNK(NT)) {
        const int na = min(TILE_CHUNK(NT), tb.natoms - ch);
        __syncthreads();
        tile_chunk_setup<P, NT, false, true>(ch, na, tb, tg, frac, base, rbeg, rpre, rec, sb, stoff, sidx, scale);
        __syncthreads();
        if (slot >= APP) continue;
        for (int at = slot; at < na; at += APP) {
            const float* r = rec + at * REC_LEN(P);
            const float w2 = r[REC_X + a] * r[REC_X + P + b];          // q_i * scale * theta_x * theta_y
            float wz[8];
            *(float4*)wz = *(const float4*)(r + REC_Z);
            *(float4*)(wz + 4) = *(const float4*)(r + REC_Z + 4);
            const int t = stoff[at];
            if (t >= 0) {
                float* rowp = tile + (t - off_ab);
                if (FIXED) {
                    // error feedback: the row's points are the differences of the ROUNDED running sum
                    // K_c = rint(sum_{j<=c} x_j), so the rounding residual of one point is carried into the
                    // next one along z and the quantisation noise is a field of tiny dipoles -- pushed to
                    // the high wavenumbers that the influence function damps
                    float run = 0.f;
                    int kprev = 0;
#pragma unroll
                    for (int c = 0; c < P; ++c) {
                        run = fmaf(w2, wz[c], run);
                        const int k = __float2int_rn(run);
                        atomicAdd((int*)rowp - c, k - kprev);
                        kprev = k;
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < P; ++c) atomicAdd(rowp - c, w2 * wz[c]);   // CAS loop: no native fp32 shared atomic
                }
            } else {
                const int4 f = sb[at];
                int gx = f.x - a; gx += gx < 0 ? K0 : 0;
                int gy = f.y - b; gy += gy < 0 ? K1 : 0;
                float* rowp = grid + ((size_t)gx * K1 + gy) * K2;
                const float w2g = w2 * inv_scale;
#pragma unroll
                for (int c = 0; c < P; ++c) {
                    int gz = f.z - c; gz += gz < 0 ? K2 : 0;
                    atomicAdd(rowp + gz, w2g * wz[c]);
                }
            }
        }
    }
    __syncthreads();
    tile_move<true, FIXED>(tile, grid, tb, tg, inv_scale);
}

template <int P, bool FORCE, int NT>
__global__ void __launch_bounds__(NT)
k_gather_tile(const float4* __restrict__ frac, const int4* __restrict__ base,
              const int* __restrict__ cell_start, TileGeom tg, const float* __restrict__ grid,
              float sx, float sy, float sz, float4* __restrict__ out)
{
    extern __shared__ __align__(16) float tile[];
    __shared__ __align__(16) float rec[TILE_CHUNK(NT) * REC_LEN(P)];
    __shared__ int4 sb[TILE_CHUNK(NT)];
    __shared__ int stoff[TILE_CHUNK(NT)], sidx[TILE_CHUNK(NT)];
    __shared__ int rbeg[TILE_MAXRANGES], rpre[TILE_MAXRANGES + 1];
    const TileBlock tb = tile_block_setup(tg, cell_start, P, rbeg, rpre);
    if (tb.natoms == 0) return;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    tile_move<false>(tile, const_cast<float*>(grid), tb, tg);
    // LPA lanes per atom, lane <-> x index a: a lane walks the P x P (y,z) plane of its x index (2 FMAs per
    // point for the z sums, 3 per row for the y sums, no idle passes), the LPA lanes of an atom are summed
    // with 4 shuffles, and 32/LPA atoms are in flight per warp.
    constexpr int LPA = P <= 4 ? 4 : 8, APW = 32 / LPA;
    const int sub = lane / LPA, a = lane % LPA;
    const bool hA = lane & (LPA / 2), hB = lane & (LPA / 4);
    const int comp = (hA ? 2 : 0) + (hB ? 1 : 0);                 // component this lane ends up holding
    const float sc_lane = comp == 0 ? -sx : (comp == 1 ? -sy : (comp == 2 ? -sz : 1.f));
    const int K0 = tg.K[0], K1 = tg.K[1], K2 = tg.K[2];
    for (int ch = 0; ch < tb.natoms; ch += TILE_CHUNK(NT)) {
        const int na = min(TILE_CHUNK(NT), tb.natoms - ch);
        __syncthreads();
        tile_chunk_setup<P, NT, FORCE>(ch, na, tb, tg, frac, base, rbeg, rpre, rec, sb, stoff, sidx);
        __syncthreads();
        for (int at0 = wid * APW; at0 < na; at0 += nw * APW) {
            const int at = at0 + sub;
            float ph = 0.f, gx_ = 0.f, gy_ = 0.f, gz_ = 0.f;
            if (at < na && a < P) {
                const float* r = rec + at * REC_LEN(P);
                float wz[8], dz[8];
                *(float4*)wz = *(const float4*)(r + REC_Z);
                *(float4*)(wz + 4) = *(const float4*)(r + REC_Z + 4);
                if (FORCE) {
                    *(float4*)dz = *(const float4*)(r + REC_DZ);
                    *(float4*)(dz + 4) = *(const float4*)(r + REC_DZ + 4);
                }
                const int toff = stoff[at];
                float pa = 0.f, gya = 0.f, gza = 0.f;             // sums over the plane: ty s0, dty s0, ty s1
                if (toff >= 0) {
                    const float* plane = tile + (toff - a * tg.XS);
#pragma unroll
                    for (int b = 0; b < P; ++b) {
                        const float* rowp = plane - b * tg.ZS;
                        float s0 = 0.f, s1 = 0.f;
#pragma unroll
                        for (int c = 0; c < P; ++c) {
                            const float v = rowp[-c];
                            s0 = fmaf(wz[c], v, s0);
                            if (FORCE) s1 = fmaf(dz[c], v, s1);
                        }
                        const float ty = r[REC_X + P + b];
                        pa = fmaf(ty, s0, pa);
                        if (FORCE) {
                            gya = fmaf(r[REC_X + 3 * P + b], s0, gya);
                            gza = fmaf(ty, s1, gza);
                        }
                    }
                } else {                                           // footprint outside the window: global grid
                    const int4 f = sb[at];
                    int gx = f.x - a; gx += gx < 0 ? K0 : 0;
                    for (int b = 0; b < P; ++b) {
                        int gy = f.y - b; gy += gy < 0 ? K1 : 0;
                        const float* rowp = grid + ((size_t)gx * K1 + gy) * K2;
                        float s0 = 0.f, s1 = 0.f;
#pragma unroll
                        for (int c = 0; c < P; ++c) {
                            int gz = f.z - c; gz += gz < 0 ? K2 : 0;
                            const float v = __ldg(rowp + gz);
                            s0 = fmaf(wz[c], v, s0);
                            if (FORCE) s1 = fmaf(dz[c], v, s1);
                        }
                        const float ty = r[REC_X + P + b];
                        pa = fmaf(ty, s0, pa);
                        if (FORCE) {
                            gya = fmaf(r[REC_X + 3 * P + b], s0, gya);
                            gza = fmaf(ty, s1, gza);
                        }
                    }
                }
                const float tx = r[REC_X + a];
                ph = tx * pa;
                if (FORCE) {
                    gx_ = r[REC_X + 2 * P + a] * pa;
                    gy_ = tx * gya;
                    gz_ = tx * gza;
                }
            }
            if (FORCE) {
                // four values over LPA lanes: the first two steps halve what a lane carries (comp above)
                float k0 = hA ? gz_ : gx_, k1 = hA ? ph : gy_;
                k0 += __shfl_xor_sync(0xffffffffu, hA ? gx_ : gz_, LPA / 2);
                k1 += __shfl_xor_sync(0xffffffffu, hA ? gy_ : ph, LPA / 2);
                float k = hB ? k1 : k0;
                k += __shfl_xor_sync(0xffffffffu, hB ? k0 : k1, LPA / 4);
#pragma unroll
                for (int o = LPA / 8; o > 0; o >>= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
                if ((lane & (LPA / 4 - 1)) == 0 && at < na) ((float*)out)[4 * sidx[at] + comp] = sc_lane * k;
            } else {
#pragma unroll
                for (int o = LPA / 2; o > 0; o >>= 1) ph += __shfl_xor_sync(0xffffffffu, ph, o);
                if (a == 0 && at < na) out[sidx[at]] = make_float4(0.f, 0.f, 0.f, ph);
            }
        }
    }
}

// -------------------------------------------------------------------------------------- one thread per atom
// The same tiles with ONE THREAD PER ATOM: the thread evaluates its atom's 3 x P spline weights into registers and
// walks all P^3 points itself.  No per-chunk weight records in shared memory, no barriers between chunks, no idle
// lanes, no shuffles: a third of the instructions of the lane-group mappings above (216 shared-memory accesses
// and as many FMAs or atomics per atom are what is left), at the price of fewer threads per block with work.
// Which atom of a chunk of up to NT a thread takes, chosen so that the lanes of a warp start on DISTINCT shared-memory
// banks.  All lanes walk their P^3 points in the same order, so the bank a lane hits at every step is (its atom's
// first-point address + a common offset) mod 32: with atoms dealt to threads as they come, a warp's 32 start banks are
// random and a shared access costs about three wavefronts.  Here atoms are bucketed by start bank (`res`, or -1 for a
// thread without an atom) and the k-th atom of a bucket goes to warp k, lane = bank; atoms beyond the NT/32-th of a
// bucket fill the slots left empty.  Returns the chunk-local index of the thread's atom or -1.  Every thread of the
// block calls it (four barriers).
template <int NT>
__device__ __forceinline__ int bank_schedule(int res)
{
    __shared__ int s_slot[NT], s_free[NT], s_left[NT], s_cnt[32], s_n[2];
    const int tid = threadIdx.x;
    s_slot[tid] = -1;
    if (tid < 32) s_cnt[tid] = 0;
    if (tid < 2) s_n[tid] = 0;
    __syncthreads();
    if (res >= 0) {
        const int k = atomicAdd(&s_cnt[res], 1);
        if (k < NT / 32) s_slot[k * 32 + res] = tid;
        else s_left[atomicAdd(&s_n[0], 1)] = tid;
    }
    __syncthreads();
    const int nleft = s_n[0];
    if (nleft > 0 && s_slot[tid] < 0) s_free[atomicAdd(&s_n[1], 1)] = tid;
    __syncthreads();
    if (tid < nleft) s_slot[s_free[tid]] = s_left[tid];
    __syncthreads();
    return s_slot[tid];
}

template <int P, bool FORCE, int NT, bool SCHED>
__global__ void __launch_bounds__(NT, 2)
k_gather_atom(const float4* __restrict__ frac, const int4* __restrict__ base, const int* __restrict__ cell_start,
              TileGeom tg, const float* __restrict__ grid, float sx, float sy, float sz, float4* __restrict__ out)
{
    extern __shared__ __align__(16) float tile[];
    __shared__ int rbeg[TILE_MAXRANGES], rpre[TILE_MAXRANGES + 1];
    const TileBlock tb = tile_block_setup(tg, cell_start, P, rbeg, rpre);
    if (tb.natoms == 0) return;
    tile_move<false>(tile, const_cast<float*>(grid), tb, tg);
    __syncthreads();
    const int K0 = tg.K[0], K1 = tg.K[1], K2 = tg.K[2];
    for (int ch = 0; ch < tb.natoms; ch += NT) {
        int li = ch + (int)threadIdx.x < tb.natoms ? (int)threadIdx.x : -1;
        if (SCHED) {
            int res = -1;
            if (li >= 0) {
                const int4 f0 = base[tile_atom(ch + li, rbeg, rpre)];
                const int ux = wrap1(f0.x - tb.o[0], K0), uy = wrap1(f0.y - tb.o[1], K1), uz = wrap1(f0.z - tb.o[2], K2);
                res = (ux * tg.XS + uy * tg.ZS + uz) & 31;
            }
            li = bank_schedule<NT>(res);
        }
        if (li < 0) continue;
        const int i = ch + li;
        const int s = tile_atom(i, rbeg, rpre);
        const float4 fw = frac[s];
        const int4 f = base[s];
        float thx[P], thy[P], thz[P], dx[P], dy[P], dz[P];
        bspline_weights<P>(fw.x, thx, dx);
        bspline_weights<P>(fw.y, thy, dy);
        bspline_weights<P>(fw.z, thz, dz);
        const int tx = wrap1(f.x - tb.o[0], K0), ty = wrap1(f.y - tb.o[1], K1), tz = wrap1(f.z - tb.o[2], K2);
        const bool in = tx >= P - 1 && tx < tg.T[0] && ty >= P - 1 && ty < tg.T[1] && tz >= P - 1 && tz < tg.T[2];
        float ph = 0.f, gx = 0.f, gy = 0.f, gz = 0.f;
        if (in) {
            const float* p0 = tile + (tx * tg.XS + ty * tg.ZS + tz);
#pragma unroll
            for (int a = 0; a < P; ++a) {
                float pa = 0.f, gya = 0.f, gza = 0.f;
#pragma unroll
                for (int b = 0; b < P; ++b) {
                    const float* rowp = p0 - a * tg.XS - b * tg.ZS;
                    float s0 = 0.f, s1 = 0.f;
#pragma unroll
                    for (int c = 0; c < P; ++c) {
                        const float v = rowp[-c];
                        s0 = fmaf(thz[c], v, s0);
                        if (FORCE) s1 = fmaf(dz[c], v, s1);
                    }
                    pa = fmaf(thy[b], s0, pa);
                    if (FORCE) { gya = fmaf(dy[b], s0, gya); gza = fmaf(thy[b], s1, gza); }
                }
                ph = fmaf(thx[a], pa, ph);
                if (FORCE) { gx = fmaf(dx[a], pa, gx); gy = fmaf(thx[a], gya, gy); gz = fmaf(thx[a], gza, gz); }
            }
        } else {                                            // footprint outside the window: global grid
            for (int a = 0; a < P; ++a) {
                int gxi = f.x - a; gxi += gxi < 0 ? K0 : 0;
                float pa = 0.f, gya = 0.f, gza = 0.f;
                for (int b = 0; b < P; ++b) {
                    int gyi = f.y - b; gyi += gyi < 0 ? K1 : 0;
                    const float* rowp = grid + ((size_t)gxi * K1 + gyi) * K2;
                    float s0 = 0.f, s1 = 0.f;
#pragma unroll
                    for (int c = 0; c < P; ++c) {
                        int gzi = f.z - c; gzi += gzi < 0 ? K2 : 0;
                        const float v = __ldg(rowp + gzi);
                        s0 = fmaf(thz[c], v, s0);
                        if (FORCE) s1 = fmaf(dz[c], v, s1);
                    }
                    pa = fmaf(thy[b], s0, pa);
                    if (FORCE) { gya = fmaf(dy[b], s0, gya); gza = fmaf(thy[b], s1, gza); }
                }
                ph = fmaf(thx[a], pa, ph);
                if (FORCE) { gx = fmaf(dx[a], pa, gx); gy = fmaf(thx[a], gya, gy); gz = fmaf(thx[a], gza, gz); }
            }
        }
        out[s] = make_float4(-sx * gx, -sy * gy, -sz * gz, ph);         // per unit charge; a-9 applies q_i
    }
}

template <int P, int NT, bool SCHED>
__global__ void __launch_bounds__(NT, 2)
k_spread_atom(const float4* __restrict__ frac, const int4* __restrict__ base, const int* __restrict__ cell_start,
              TileGeom tg, float* __restrict__ grid)
{
    extern __shared__ __align__(16) float tile[];
    __shared__ int rbeg[TILE_MAXRANGES], rpre[TILE_MAXRANGES + 1];
    __shared__ float s_part[NT / 32];
    const TileBlock tb = tile_block_setup(tg, cell_start, P, rbeg, rpre);
    if (tb.natoms == 0) return;
    const int K0 = tg.K[0], K1 = tg.K[1], K2 = tg.K[2];
    const int tsize = tg.XS * tg.T[0];
    for (int e = threadIdx.x; e < (tsize >> 2); e += NT) ((float4*)tile)[e] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (threadIdx.x < (tsize & 3)) tile[(tsize & ~3) + threadIdx.x] = 0.f;
    // fixed-point scale of the block (see k_spread_tile): |tile point| <= (2/3)^3 sum |q|
    float aq = 0.f;
    for (int i = threadIdx.x; i < tb.natoms; i += NT) aq += fabsf(frac[tile_atom(i, rbeg, rpre)].w);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) aq += __shfl_xor_sync(0xffffffffu, aq, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = aq;
    __syncthreads();
    aq = 0.f;
#pragma unroll
    for (int k = 0; k < NT / 32; ++k) aq += s_part[k];
    const float scale = aq > 0.f ? 1073741824.f / (0.2962963f * aq * 1.0001f) : 1.f;
    const float inv_scale = 1.f / scale;
    for (int ch = 0; ch < tb.natoms; ch += NT) {
        int li = ch + (int)threadIdx.x < tb.natoms ? (int)threadIdx.x : -1;
        if (SCHED) {
            int res = -1;
            if (li >= 0) {
                const int4 f0 = base[tile_atom(ch + li, rbeg, rpre)];
                const int ux = wrap1(f0.x - tb.o[0], K0), uy = wrap1(f0.y - tb.o[1], K1), uz = wrap1(f0.z - tb.o[2], K2);
                res = (ux * tg.XS + uy * tg.ZS + uz) & 31;
            }
            li = bank_schedule<NT>(res);
        }
        if (li < 0) continue;
        const int i = ch + li;
        const int s = tile_atom(i, rbeg, rpre);
        const float4 fw = frac[s];
        const int4 f = base[s];
        float thx[P], thy[P], thz[P], dd[P];
        bspline_weights<P>(fw.x, thx, dd);
        bspline_weights<P>(fw.y, thy, dd);
        bspline_weights<P>(fw.z, thz, dd);
        const float qs = fw.w * scale;
#pragma unroll
        for (int a = 0; a < P; ++a) thx[a] *= qs;
        const int tx = wrap1(f.x - tb.o[0], K0), ty = wrap1(f.y - tb.o[1], K1), tz = wrap1(f.z - tb.o[2], K2);
        const bool in = tx >= P - 1 && tx < tg.T[0] && ty >= P - 1 && ty < tg.T[1] && tz >= P - 1 && tz < tg.T[2];
        if (in) {
            int* p0 = (int*)tile + (tx * tg.XS + ty * tg.ZS + tz);
#pragma unroll
            for (int a = 0; a < P; ++a)
#pragma unroll
                for (int b = 0; b < P; ++b) {
                    int* rowp = p0 - a * tg.XS - b * tg.ZS;
                    const float w2 = thx[a] * thy[b];
                    // error feedback along z: the row's points are the differences of the ROUNDED running sum
                    float run = 0.f;
                    int kprev = 0;
#pragma unroll
                    for (int c = 0; c < P; ++c) {
                        run = fmaf(w2, thz[c], run);
                        const int k = __float2int_rn(run);
                        atomicAdd(rowp - c, k - kprev);
                        kprev = k;
                    }
                }
        } else {
            for (int a = 0; a < P; ++a) {
                int gxi = f.x - a; gxi += gxi < 0 ? K0 : 0;
                for (int b = 0; b < P; ++b) {
                    int gyi = f.y - b; gyi += gyi < 0 ? K1 : 0;
                    float* rowp = grid + ((size_t)gxi * K1 + gyi) * K2;
                    const float w2g = thx[a] * thy[b] * inv_scale;
#pragma unroll
                    for (int c = 0; c < P; ++c) {
                        int gzi = f.z - c; gzi += gzi < 0 ? K2 : 0;
                        atomicAdd(rowp + gzi, w2g * thz[c]);
                    }
                }
            }
        }
    }
    __syncthreads();
    tile_move<true, true>(tile, grid, tb, tg, inv_scale);
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
        // fused x-axis pass: needs K0 = 2^a 3^b 5^c; then the 3-D transforms become batched 2-D cuFFT transforms over
        // (y,z) around k_xline_influence
        if (ctx->xf_ok) { cufftDestroy(ctx->plan2_r2c); cufftDestroy(ctx->plan2_c2r); ctx->xf_ok = false; }
        ctx->fft3_ok = false;
        {
            int r = grid[0], np = 0;
            int radix[XF_MAXPASS];
            while (r % 4 == 0 && np < XF_MAXPASS) { radix[np++] = 4; r /= 4; }
            for (int pfac : {2, 3, 5}) while (r % pfac == 0 && np < XF_MAXPASS) { radix[np++] = pfac; r /= pfac; }
            const size_t sm = sizeof(float2) * ((size_t)grid[0] * (2 * XF_TJ + 1));
            if (r == 1 && sm <= 200 * 1024) {
                int nn[2] = {grid[1], grid[2]};
                const int K2h = grid[2] / 2 + 1;
                cufftResult r1 = cufftPlanMany(&ctx->plan2_r2c, 2, nn, nullptr, 1, grid[1] * grid[2], nullptr, 1, grid[1] * K2h,
                                               CUFFT_R2C, grid[0]);
                cufftResult r2 = r1 == CUFFT_SUCCESS ? cufftPlanMany(&ctx->plan2_c2r, 2, nn, nullptr, 1, grid[1] * K2h, nullptr, 1,
                                                                     grid[1] * grid[2], CUFFT_C2R, grid[0]) : r1;
                if (r1 == CUFFT_SUCCESS && r2 != CUFFT_SUCCESS) cufftDestroy(ctx->plan2_r2c);
                if (r1 == CUFFT_SUCCESS && r2 == CUFFT_SUCCESS) {
                    ctx->xf_ok = true;
                    ctx->xf_npass = np;
                    for (int k = 0; k < np; ++k) ctx->xf_radix[k] = radix[k];
                    // roots of unity e^{-2 pi i m/K} of the three axes, one after the other
                    std::vector<float2> W;
                    for (int d = 0; d < 3; ++d)
                        for (int m = 0; m < grid[d]; ++m) {
                            const double a = -2.0 * M_PI * (double)m / (double)grid[d];
                            W.push_back(make_float2((float)cos(a), (float)sin(a)));
                        }
                    ctx->fft3_ok = xline2_supported(grid[0]) && xline2_supported(grid[1]) && zline_supported(grid[2]);
                    SQEQ_TRY(sqeq_reserve(ctx, ctx->xf_tw, sizeof(float2) * W.size()));
                    CUDA_TRY(ctx, cudaMemcpy(ctx->xf_tw.p, W.data(), sizeof(float2) * W.size(), cudaMemcpyHostToDevice));
                }
            }
        }
        for (int d = 0; d < 3; ++d) ctx->K[d] = grid[d];
        const size_t G3 = (size_t)grid[0] * grid[1] * grid[2];
        const size_t S3 = (size_t)grid[0] * grid[1] * (grid[2] / 2 + 1);
        SQEQ_TRY(sqeq_reserve(ctx, ctx->grid, sizeof(float) * G3));
        SQEQ_TRY(sqeq_reserve(ctx, ctx->spec, sizeof(float2) * S3));
    }
    // per-axis tables (DESIGN.md R-PME), evaluated in fp64 and stored as fp32:
    //   Bg[m] = |b(m)|^2 exp(-pi^2 mt^2/alpha^2),  s[m] = mt^2
    const int Ksum = grid[0] + grid[1] + grid[2];
    std::vector<float> tab(2 * (size_t)Ksum);
    size_t off = 0;
    for (int d = 0; d < 3; ++d) {
        const int K = grid[d];
        float* Bg = tab.data() + off; float* s = Bg + K;
        for (int m = 0; m < K; ++m) {
            double re = 0, im = 0;
            for (int k = 0; k <= order - 2; ++k) {
                double a = 2.0 * M_PI * (double)m * (double)k / (double)K;
                double M = host_bspline(order, (double)(k + 1));
                re += M * cos(a);
                im += M * sin(a);
            }
            double mp = (m <= K / 2 ? m : m - K) / box[d];
            s[m] = (float)(mp * mp);
            // odd order: the sum is exactly zero on the Nyquist plane; that plane is left out (reading G19)
            const bool nyq_odd = (order & 1) && 2 * m == K;
            Bg[m] = nyq_odd ? 0.f : (float)(exp(-M_PI * M_PI * mp * mp / (alpha * alpha)) / (re * re + im * im));
        }
        off += 2 * (size_t)K;
    }
    SQEQ_TRY(sqeq_reserve(ctx, ctx->tabs, sizeof(float) * tab.size()));
    CUDA_TRY(ctx, cudaMemcpy(ctx->tabs.p, tab.data(), sizeof(float) * tab.size(), cudaMemcpyHostToDevice));
    ctx->order = order;
    ctx->tab_alpha = alpha;
    for (int d = 0; d < 3; ++d) ctx->tab_box[d] = box[d];
    return SQEQ_OK;
}

// Chooses the cell group and tile shape for the shared-memory spread/gather kernels; false when the
// geometry does not suit them (window wider than the grid, no list) and the global kernels run.
static bool plan_tiles(const sqeq_ctx* ctx, const sqeq_nlist* nl, int P, TileGeom& best, size_t& best_bytes,
                       int& best_nt)
{
    if (!nl || !nl->cell_start || ctx->pme_tiles_off) return false;
    if (ctx->K[2] % 4 != 0) return false;                 // float4 window rows
    const int M = 1;
    double best_cost = 1e300;
    bool found = false;
    const int64_t want_groups = 2 * (int64_t)ctx->sm_count;
    for (int pass = 0; pass < 2 && !found; ++pass)       // pass 1 drops the "enough blocks" wish
        for (int nt = 256; nt <= 512; nt *= 2) {
            static const int force_nt = getenv("SQEQ_TILE_NT") ? atoi(getenv("SQEQ_TILE_NT")) : 0;
            if (force_nt && nt != force_nt) continue;
            // 227 KB per SM: four 256-thread blocks or two 512-thread blocks, records included
            static const int force_blocks = getenv("SQEQ_TILE_BLOCKS") ? atoi(getenv("SQEQ_TILE_BLOCKS")) : 0;
            const int blocks_per_sm = force_blocks ? force_blocks : (nt == 256 ? 4 : 2);
            const size_t limit = (size_t)(224 * 1024 / blocks_per_sm) - (size_t)(nt / 4) * (REC_LEN(P) * 4 + 24) - 256;
            for (int gxy = 1; gxy <= 4; ++gxy)
                for (int gz = 1; gz <= 12; ++gz) {
                    TileGeom tg;
                    const int g[3] = {gxy, gxy, gz};
                    bool ok = true;
                    int64_t groups = 1;
                    for (int d = 0; d < 3; ++d) {
                        tg.K[d] = ctx->K[d];
                        tg.nc[d] = nl->ncell[d];
                        tg.g[d] = g[d] < tg.nc[d] ? g[d] : tg.nc[d];
                        tg.ng[d] = (tg.nc[d] + tg.g[d] - 1) / tg.g[d];
                        tg.T[d] = (int)(((int64_t)tg.g[d] * tg.K[d]) / tg.nc[d]) + 2 + 2 * M + (P - 1);
                        if (d == 2) tg.T[d] = (tg.T[d] + 3 + 3) & ~3;     // origin rounded down to 4, extent up
                        if (tg.T[d] > tg.K[d] || tg.T[d] > 1023) ok = false;
                        groups *= tg.ng[d];
                    }
                    if (!ok || tg.g[0] * tg.g[1] > TILE_MAXRANGES) continue;
                    if (tg.T[0] * tg.T[1] >= 65536) continue;
                    if (pass == 0 && groups < want_groups) continue;
                    tg.M = M;
                    tg.T1_magic = (unsigned)((0x100000000ull + tg.T[1] - 1) / tg.T[1]);
                    tg.nvz_magic = (unsigned)((0x100000000ull + tg.T[2] / 4 - 1) / (tg.T[2] / 4));
                    if ((uint64_t)tg.T[0] * tg.T[1] * (tg.T[2] / 4) * (tg.T[2] / 4) >= 0x100000000ull) continue;   // magic division exact
                    // strides: smallest padding that puts the 32 rows (a,b) of a full pass in distinct banks
                    const int nrow = (P * P >= 32) ? 32 : 0;
                    int bz = -1, bx = -1;
                    for (int zs = tg.T[2]; zs < tg.T[2] + 32 && bz < 0; ++zs)
                        for (int xs = tg.T[1] * zs; xs < tg.T[1] * zs + 32; ++xs) {
                            unsigned seen = 0;
                            bool distinct = true;
                            for (int r = 0; r < nrow; ++r) {
                                const int bank = (((-(r / P) * xs - (r % P) * zs) % 32) + 32) % 32;
                                if (seen & (1u << bank)) { distinct = false; break; }
                                seen |= 1u << bank;
                            }
                            if (distinct) { bz = zs; bx = xs; break; }
                        }
                    if (bz < 0) { bz = tg.T[2]; bx = tg.T[1] * tg.T[2]; }
                    tg.ZS = bz; tg.XS = bx;
                    const size_t bytes = sizeof(float) * (size_t)tg.XS * tg.T[0];
                    if (bytes > limit) continue;
                    // window points moved per cell, plus a charge for idle SMs when blocks are few
                    double cost = (double)tg.T[0] * tg.T[1] * tg.T[2] / ((double)tg.g[0] * tg.g[1] * tg.g[2]);
                    const double slots = (double)ctx->sm_count * blocks_per_sm;
                    const double waves = (double)groups / slots;
                    cost *= ceil(waves) / waves;
                    if (cost < best_cost) { best_cost = cost; best = tg; best_bytes = bytes; best_nt = nt; found = true; }
                }
        }
    return found;
}

template <int P>
static int pme_run_t(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3], bool want_force,
                     bool want_energy, cudaStream_t st)
{
    // the tile plan depends only on (cells of the list, grid, order): searched once, then reused
    static_assert(sizeof(TileGeom) <= sizeof(ctx->tile_plan.blob), "tile plan cache too small");
    TileGeom tg;
    size_t tile_bytes = 0;
    int nt = 256;
    bool tiles;
    {
        auto& tp = ctx->tile_plan;
        const bool same = tp.valid && nl && tp.order == P && tp.K[0] == ctx->K[0] && tp.K[1] == ctx->K[1] && tp.K[2] == ctx->K[2] &&
                          tp.nc[0] == nl->ncell[0] && tp.nc[1] == nl->ncell[1] && tp.nc[2] == nl->ncell[2];
        if (same) {
            memcpy(&tg, tp.blob, sizeof(TileGeom));
            tile_bytes = tp.bytes; nt = tp.nt; tiles = tp.tiles;
        } else {
            tiles = plan_tiles(ctx, nl, P, tg, tile_bytes, nt);
            if (nl) {
                memcpy(tp.blob, &tg, sizeof(TileGeom));
                tp.bytes = tile_bytes; tp.nt = nt; tp.tiles = tiles; tp.order = P; tp.valid = true;
                for (int d = 0; d < 3; ++d) { tp.K[d] = ctx->K[d]; tp.nc[d] = nl->ncell[d]; }
            }
        }
    }
    const int ngroups = tiles ? tg.ng[0] * tg.ng[1] * tg.ng[2] : 0;
    // one thread per atom needs many blocks to hide its long serial chains (measured: faster from cfg 3's 343 tiles
    // on, slower at cfg 1/2's 64 and 125): lane groups below two tiles per SM
    const bool atom_threads = ctx->pme_atom_threads == 2 || (ctx->pme_atom_threads == 1 && ngroups >= 2 * ctx->sm_count);
    const bool atom_sched = ctx->pme_atom_sched == 2 || (ctx->pme_atom_sched == 1 && ngroups >= 4 * ctx->sm_count);
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
        if (tiles && atom_threads && !ctx->spread_float) {
            // lanes dealt by start bank where tiles are many (cfg 4: 1000 tiles, -8 us per evaluation; cfg 3: 343 tiles,
            // +4 us from the four extra barriers)
            auto kern = atom_sched ? k_spread_atom<P, PME_ATOM_NT, true> : k_spread_atom<P, PME_ATOM_NT, false>;
            CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_bytes));
            kern<<<ngroups, PME_ATOM_NT, tile_bytes, st>>>(frac, base, nl->cell_start, tg, grid);
        } else if (tiles) {
            auto kern = ctx->spread_float ? (nt == 256 ? k_spread_tile<P, 256, false> : k_spread_tile<P, 512, false>)
                                          : (nt == 256 ? k_spread_tile<P, 256, true> : k_spread_tile<P, 512, true>);
            CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_bytes));
            kern<<<ngroups, nt, tile_bytes, st>>>(frac, base, nl->cell_start, tg, grid);
        } else {
            k_spread<P><<<ceil_div(n, SPREAD_APB), 256, 0, st>>>(n, frac, base, K0, K1, K2, grid);
        }
        KERNEL_CHECK(ctx);
    }
    if (ctx->gridQ.p) SQEQ_TRY(sqeq_reserve(ctx, ctx->gridQ, sizeof(float) * G3));    // the grid may have grown since the capture was enabled
    if (ctx->gridQ.p) CUDA_TRY(ctx, cudaMemcpyAsync(ctx->gridQ.p, grid, sizeof(float) * G3, cudaMemcpyDeviceToDevice, st));
    const bool fused = ctx->xf_ok && !ctx->fft_fused_off;
    // E_rec accumulator: cleared here rather than next to its kernel so that the transform kernels follow one another
    // in the stream (programmatic dependent launch needs the kernels adjacent)
    CUDA_TRY(ctx, cudaMemsetAsync((double*)ctx->scal.p + 1, 0, sizeof(double), st));
    // all three axes by the two-step kernels of fftx.cu / fftz.cu (no cuFFT call) where the extents allow
    const bool own3 = fused && ctx->fft3_ok && !ctx->fft_xline2_off && !ctx->fft_own_off;
    const float2* Wx = (const float2*)ctx->xf_tw.p;
    const float2* Wy = Wx + K0;
    const float2* Wz = Wy + K1;
    if (own3) {
        StageTimer tm(ctx, SQEQ_T_FFT_FWD, st);
        SQEQ_TRY(zline_run(ctx, K0 * K1, K2, Wz, grid, spec, false, st));
        KERNEL_CHECK(ctx);
        SQEQ_TRY(yline_run(ctx, K0, K1, K2h, Wy, spec, false, st));
        KERNEL_CHECK(ctx);
    } else {
        StageTimer tm(ctx, SQEQ_T_FFT_FWD, st);
        cufftHandle plan = fused ? ctx->plan2_r2c : ctx->plan_r2c;
        cufftSetStream(plan, st);
        cufftResult r = cufftExecR2C(plan, grid, (cufftComplex*)spec);
        if (r != CUFFT_SUCCESS) return sqeq_fail(ctx, SQEQ_ECUFFT, "cufftExecR2C failed: %d", (int)r);
    }
    {
        StageTimer tm(ctx, SQEQ_T_INFLUENCE, st);
        double* e_out = (double*)ctx->scal.p + 1;
        const float inv_piV = (float)(1.0 / (M_PI * box[0] * box[1] * box[2]));
        if (fused) {
            // forward x-transform, influence multiply + energy, inverse x-transform: one pass over the spectrum
            if (!ctx->fft_xline2_off && xline2_supported(K0)) {
                SQEQ_TRY(xline2_run(ctx, K0, K1, K2h, K2, (const float*)ctx->tabs.p, inv_piV, (const float2*)ctx->xf_tw.p, spec,
                                    e_out, st));
            } else {
            XfPlan pl;
            pl.N = K0; pl.npass = ctx->xf_npass;
            for (int k = 0; k < pl.npass; ++k) pl.radix[k] = ctx->xf_radix[k];
            const size_t sm = sizeof(float2) * ((size_t)K0 * (2 * XF_TJ + 1));
            CUDA_TRY(ctx, cudaFuncSetAttribute(k_xline_influence, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            k_xline_influence<<<ceil_div((int64_t)K1 * K2h, XF_TJ), XF_NT, sm, st>>>(pl, K1, K2h, K2, (const float*)ctx->tabs.p, inv_piV,
                                                                                    (const float2*)ctx->xf_tw.p, spec, e_out);
            }
        } else {
            int nb = ceil_div((int64_t)K0 * K1, 8);
            if (nb > ctx->sm_count * 8) nb = ctx->sm_count * 8;
            k_influence<<<nb, 256, 0, st>>>(K0, K1, K2h, K2, (const float*)ctx->tabs.p, inv_piV, spec, e_out);
        }
        KERNEL_CHECK(ctx);
    }
    if (own3) {
        StageTimer tm(ctx, SQEQ_T_FFT_INV, st);
        SQEQ_TRY(yline_run(ctx, K0, K1, K2h, Wy, spec, true, st));
        KERNEL_CHECK(ctx);
        SQEQ_TRY(zline_run(ctx, K0 * K1, K2, Wz, grid, spec, true, st));
        KERNEL_CHECK(ctx);
    } else {
        StageTimer tm(ctx, SQEQ_T_FFT_INV, st);
        cufftHandle plan = fused ? ctx->plan2_c2r : ctx->plan_c2r;
        cufftSetStream(plan, st);
        cufftResult r = cufftExecC2R(plan, (cufftComplex*)spec, grid);
        if (r != CUFFT_SUCCESS) return sqeq_fail(ctx, SQEQ_ECUFFT, "cufftExecC2R failed: %d", (int)r);
    }
    {
        StageTimer tm(ctx, SQEQ_T_GATHER, st);
        const float sx = (float)(K0 / box[0]), sy = (float)(K1 / box[1]), sz = (float)(K2 / box[2]);
        float4* rec = (float4*)ctx->rec_out.p;
        if (tiles && atom_threads) {
            auto kern = atom_sched ? (want_force ? k_gather_atom<P, true, PME_ATOM_NT, true> : k_gather_atom<P, false, PME_ATOM_NT, true>)
                                   : (want_force ? k_gather_atom<P, true, PME_ATOM_NT, false> : k_gather_atom<P, false, PME_ATOM_NT, false>);
            CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_bytes));
            kern<<<ngroups, PME_ATOM_NT, tile_bytes, st>>>(frac, base, nl->cell_start, tg, grid, sx, sy, sz, rec);
        } else if (tiles) {
            auto kern = want_force ? (nt == 256 ? k_gather_tile<P, true, 256> : k_gather_tile<P, true, 512>)
                                   : (nt == 256 ? k_gather_tile<P, false, 256> : k_gather_tile<P, false, 512>);
            CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_bytes));
            kern<<<ngroups, nt, tile_bytes, st>>>(frac, base, nl->cell_start, tg, grid, sx, sy, sz, rec);
        } else if (want_force)
            k_gather<P, true><<<nbw, 256, 0, st>>>(n, frac, base, K0, K1, K2, grid, sx, sy, sz, rec);
        else
            k_gather<P, false><<<nbw, 256, 0, st>>>(n, frac, base, K0, K1, K2, grid, sx, sy, sz, rec);
        KERNEL_CHECK(ctx);
    }
    (void)want_energy;
    return SQEQ_OK;
}

int pme_run(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3], bool want_force,
            bool want_energy, cudaStream_t st)
{
    switch (ctx->order) {
        case 4: return pme_run_t<4>(ctx, nl, n, box, want_force, want_energy, st);
        case 5: return pme_run_t<5>(ctx, nl, n, box, want_force, want_energy, st);
        case 6: return pme_run_t<6>(ctx, nl, n, box, want_force, want_energy, st);
        case 7: return pme_run_t<7>(ctx, nl, n, box, want_force, want_energy, st);
        case 8: return pme_run_t<8>(ctx, nl, n, box, want_force, want_energy, st);
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
