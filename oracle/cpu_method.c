/* oracle/cpu_method.c
 *
 * TEST / BENCH INFRASTRUCTURE -- NOT THE PARITY ORACLE AND NOT PART OF THE PRODUCT PATH.
 * A CPU RESTATEMENT OF THE METHOD itself (arxiv 2503.21176 sections 3.1-3.3): cell-list neighbour search
 * (PAPER.md:43-71), real-space erfc sum over the list (Eq. 3), smooth PME spreading and gathering
 * (Alg. 2 steps 1 and 5) -- fp64, OpenMP.  The FFTs and the influence multiply are done by the
 * Python side (cpu_method.py: numpy.fft = pocketfft).  bench.py times it as the second CPU baseline ("kind":
 * "method_cpu"): what the same algorithm costs on the box's host cores, next to the deliberately slow O(N^2)
 * oracle.  It is pinned AGAINST the oracle (tests/test_oracle_pins.py) and shares no code with it or with csrc/.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int cm_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* wrapped coordinates in [0, L) and cell index; cells of edge >= rl (nc = floor(L / rl) >= 3 per axis required) */
static inline double wrap(double x, double L)
{
    double w = x - floor(x / L) * L;
    return w >= L ? w - L : w;
}

/* Counting sort of the atoms by cell: order[s] = atom index of the s-th atom in cell-major order,
 * cell_start[ncells + 1].  xw[n][3] receives the wrapped positions (caller order). */
void cm_bin(int64_t n, const double *pos, const double box[3], const int nc[3], double *xw, int32_t *cell_of,
            int64_t *cell_start, int32_t *order)
{
    const int64_t ncells = (int64_t)nc[0] * nc[1] * nc[2];
    memset(cell_start, 0, sizeof(int64_t) * (ncells + 1));
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int c[3];
        for (int d = 0; d < 3; ++d) {
            double w = wrap(pos[3 * i + d], box[d]);
            xw[3 * i + d] = w;
            int k = (int)(w / box[d] * nc[d]);
            c[d] = k >= nc[d] ? nc[d] - 1 : k;
        }
        cell_of[i] = (c[0] * nc[1] + c[1]) * nc[2] + c[2];
    }
    for (int64_t i = 0; i < n; ++i) cell_start[cell_of[i] + 1]++;
    for (int64_t c = 0; c < ncells; ++c) cell_start[c + 1] += cell_start[c];
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * ncells);
    memcpy(fill, cell_start, sizeof(int64_t) * ncells);
    for (int64_t i = 0; i < n; ++i) order[fill[cell_of[i]]++] = (int32_t)i;
    free(fill);
}

/* Directed neighbour rows (every pair from both sides), two passes with the same loop: count (col == NULL) and
 * fill.  A pair is listed when the minimum-image distance of the WRAPPED positions is below rl; shift[3] is the
 * image of j (in box lengths, relative to the wrapped positions) that is the near one. */
void cm_rows(int64_t n, const double *xw, const double box[3], const int nc[3], double rl, const int32_t *cell_of,
             const int64_t *cell_start, const int32_t *order, int64_t *row_ptr, int32_t *col, int8_t *shift)
{
    const double rr = rl * rl;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        const int cid = cell_of[i];
        const int cz = cid % nc[2], cy = (cid / nc[2]) % nc[1], cx = cid / (nc[2] * nc[1]);
        int64_t cnt = 0, o = col ? row_ptr[i] : 0;
        for (int ox = -1; ox <= 1; ++ox)
            for (int oy = -1; oy <= 1; ++oy)
                for (int oz = -1; oz <= 1; ++oz) {
                    int ux = cx + ox, uy = cy + oy, uz = cz + oz, sx = 0, sy = 0, sz = 0;
                    if (ux < 0) { ux += nc[0]; sx = -1; } else if (ux >= nc[0]) { ux -= nc[0]; sx = 1; }
                    if (uy < 0) { uy += nc[1]; sy = -1; } else if (uy >= nc[1]) { uy -= nc[1]; sy = 1; }
                    if (uz < 0) { uz += nc[2]; sz = -1; } else if (uz >= nc[2]) { uz -= nc[2]; sz = 1; }
                    const int64_t c = ((int64_t)ux * nc[1] + uy) * nc[2] + uz;
                    for (int64_t t = cell_start[c]; t < cell_start[c + 1]; ++t) {
                        const int32_t j = order[t];
                        if (j == i) continue;
                        const double dx = xw[3 * j] + sx * box[0] - xw[3 * i];
                        const double dy = xw[3 * j + 1] + sy * box[1] - xw[3 * i + 1];
                        const double dz = xw[3 * j + 2] + sz * box[2] - xw[3 * i + 2];
                        if (dx * dx + dy * dy + dz * dz < rr) {
                            if (col) {
                                col[o] = j;
                                shift[3 * o] = (int8_t)sx; shift[3 * o + 1] = (int8_t)sy; shift[3 * o + 2] = (int8_t)sz;
                                ++o;
                            }
                            ++cnt;
                        }
                    }
                }
        if (!col) row_ptr[i + 1] = cnt;
    }
    if (!col) {
        row_ptr[0] = 0;
        for (int64_t i = 0; i < n; ++i) row_ptr[i + 1] += row_ptr[i];
    }
}

/* Real-space sum over the rows at the CURRENT wrapped-image positions x (= pos - build-time wrap count * L, so the
 * list's shifts stay valid on a stale list): pairs with r < rc only. */
void cm_realspace(int64_t n, const double *x, const double *q, const double box[3], double rc, double alpha,
                  const int64_t *row_ptr, const int32_t *col, const int8_t *shift, double *phi, double *F)
{
    const double rr = rc * rc, c2 = 2.0 * alpha / sqrt(3.14159265358979323846);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        double p = 0.0, fx = 0.0, fy = 0.0, fz = 0.0;
        for (int64_t o = row_ptr[i]; o < row_ptr[i + 1]; ++o) {
            const int32_t j = col[o];
            const double dx = x[3 * i] - x[3 * j] - shift[3 * o] * box[0];
            const double dy = x[3 * i + 1] - x[3 * j + 1] - shift[3 * o + 1] * box[1];
            const double dz = x[3 * i + 2] - x[3 * j + 2] - shift[3 * o + 2] * box[2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (!(r2 < rr)) continue;
            const double r = sqrt(r2);
            const double t = erfc(alpha * r) / r;
            const double g = q[j] * (t + c2 * exp(-alpha * alpha * r2)) / r2;
            p += q[j] * t;
            fx += g * dx; fy += g * dy; fz += g * dz;
        }
        phi[i] = p;
        F[3 * i] = q[i] * fx; F[3 * i + 1] = q[i] * fy; F[3 * i + 2] = q[i] * fz;
    }
}

/* cardinal B-spline weights M_p(w + j), j = 0..p-1, and their derivatives, by the recursion */
static void weights(int p, double w, double *th, double *dth)
{
    double a[16];
    for (int j = 0; j < p; ++j) a[j] = 0.0;
    a[0] = w; a[1] = 1.0 - w;
    for (int n = 3; n <= p; ++n) {
        if (n == p)
            for (int j = 0; j < p; ++j) dth[j] = a[j] - (j > 0 ? a[j - 1] : 0.0);
        for (int j = n - 1; j >= 0; --j) {
            const double lo = j > 0 ? a[j - 1] : 0.0;
            a[j] = ((w + j) * a[j] + (n - w - j) * lo) / (n - 1);
        }
    }
    for (int j = 0; j < p; ++j) th[j] = a[j];
}

/* Spreading: thread-private grids, summed at the end.  Q[K0][K1][K2]. */
void cm_spread(int64_t n, const double *pos, const double *q, const double box[3], const int K[3], int p, double *Q)
{
    const int64_t G = (int64_t)K[0] * K[1] * K[2];
    const int nth = cm_num_threads();
    double *priv = (double *)calloc((size_t)nth * G, sizeof(double));
#pragma omp parallel
    {
#ifdef _OPENMP
        double *g = priv + (size_t)omp_get_thread_num() * G;
#else
        double *g = priv;
#endif
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double th[3][16], dth[16];
            int f[3];
            for (int d = 0; d < 3; ++d) {
                double u = pos[3 * i + d] / box[d];
                u = (u - floor(u)) * K[d];
                int fi = (int)u;
                if (fi >= K[d]) { fi -= K[d]; u -= K[d]; }
                weights(p, u - fi, th[d], dth);
                f[d] = fi;
            }
            for (int a = 0; a < p; ++a) {
                const int gx = (f[0] - a + K[0]) % K[0];
                for (int b = 0; b < p; ++b) {
                    const int gy = (f[1] - b + K[1]) % K[1];
                    const double w2 = q[i] * th[0][a] * th[1][b];
                    double *row = g + ((int64_t)gx * K[1] + gy) * K[2];
                    for (int c = 0; c < p; ++c) row[(f[2] - c + K[2]) % K[2]] += w2 * th[2][c];
                }
            }
        }
#pragma omp for schedule(static)
        for (int64_t k = 0; k < G; ++k) {
            double s = 0.0;
            for (int t = 0; t < nth; ++t) s += priv[(size_t)t * G + k];
            Q[k] = s;
        }
    }
    free(priv);
}

/* Gathering from the potential grid Phi: phi_i and F_i = -q_i (K/L) sum dW Phi */
void cm_gather(int64_t n, const double *pos, const double *q, const double box[3], const int K[3], int p,
               const double *Phi, double *phi, double *F)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double th[3][16], dth[3][16];
        int f[3];
        for (int d = 0; d < 3; ++d) {
            double u = pos[3 * i + d] / box[d];
            u = (u - floor(u)) * K[d];
            int fi = (int)u;
            if (fi >= K[d]) { fi -= K[d]; u -= K[d]; }
            weights(p, u - fi, th[d], dth[d]);
            f[d] = fi;
        }
        double ph = 0.0, gx_ = 0.0, gy_ = 0.0, gz_ = 0.0;
        for (int a = 0; a < p; ++a) {
            const int gx = (f[0] - a + K[0]) % K[0];
            for (int b = 0; b < p; ++b) {
                const int gy = (f[1] - b + K[1]) % K[1];
                const double *row = Phi + ((int64_t)gx * K[1] + gy) * K[2];
                double s0 = 0.0, s1 = 0.0;
                for (int c = 0; c < p; ++c) {
                    const double v = row[(f[2] - c + K[2]) % K[2]];
                    s0 += th[2][c] * v;
                    s1 += dth[2][c] * v;
                }
                ph += th[0][a] * th[1][b] * s0;
                gx_ += dth[0][a] * th[1][b] * s0;
                gy_ += th[0][a] * dth[1][b] * s0;
                gz_ += th[0][a] * th[1][b] * s1;
            }
        }
        phi[i] = ph;
        F[3 * i] = -q[i] * K[0] / box[0] * gx_;
        F[3 * i + 1] = -q[i] * K[1] / box[1] * gy_;
        F[3 * i + 2] = -q[i] * K[2] / box[2] * gz_;
    }
}
