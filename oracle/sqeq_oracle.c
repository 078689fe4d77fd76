/* oracle/sqeq_oracle.c
 *
 * TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT PATH.
 * Plain, slow, fp64 CPU implementation of the periodic Coulomb evaluation of
 * arxiv 2503.21176 ("GPU-Accelerated Charge-Equilibration for Shadow Molecular
 * Dynamics in Python"): brute-force minimum-image neighbour search, the
 * erfc-screened real-space sum, direct (regular) Ewald summation, and smooth
 * Particle Mesh Ewald.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code with
 * the CUDA path under paper_2503_21176_b200/csrc/ and is never linked into it.
 *
 * Citations: PAPER.md:N = line N of /root/reference/PAPER.md.
 *   Eq. 1-5   PAPER.md:75-94   Coulomb energy and its Ewald split
 *   Alg. 1    PAPER.md:59-71   neighbour list (the cell method reaches the set
 *                              that the O(N^2) definition below writes out)
 *   Alg. 2    PAPER.md:140-151 smooth PME, five steps
 * Where the paper is silent (spline conventions, FFT normalisation, strict
 * cutoff, ...) the reading is the one listed in DESIGN.md section 3.
 *
 * Everything is fp64, written in the order of the definitions; there is no
 * blocking, no cell list, no FFT butterflies (the 3-D DFT is a sum of naive
 * 1-D line DFTs).  OpenMP only distributes independent outer iterations.
 * Compile with -ffp-contract=off so that the cutoff predicate is evaluated
 * with individually rounded IEEE operations (DESIGN.md R-NL).
 *
 * Units: k_e = 1 (charges in e, lengths in Angstrom, potential e/A, energy
 * e^2/A).  Boxes are orthorhombic: box[3] = edge lengths.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------ */
/* c-NL: minimum-image pair predicate ("minimum image            */
/* convention", "within the cutoff range"; strict '<', DESIGN.md R-NL).      */
/*   d_k = pos[j][k] - pos[i][k]          (raw, unwrapped positions)         */
/*   s_k = -rint(d_k / L_k);  d_k = d_k + s_k * L_k                          */
/*   r2  = (d_x*d_x + d_y*d_y) + d_z*d_z ;   in range  <=>  r2 < r*r         */
/* Returns 1 if in range; writes the shift s (so that r_j + s*L - r_i = d),  */
/* the minimum-image vector d and r2.                                        */
/* ------------------------------------------------------------------------ */
static int orc_pair(const double *pi, const double *pj, const double box[3],
                    double rr, int s[3], double d[3], double *r2out)
{
    for (int k = 0; k < 3; ++k) {
        double dk = pj[k] - pi[k];
        double sk = -rint(dk / box[k]);
        double sl = sk * box[k];
        dk = dk + sl;
        d[k] = dk;
        s[k] = (int)sk;
    }
    double xx = d[0] * d[0];
    double yy = d[1] * d[1];
    double zz = d[2] * d[2];
    double r2 = (xx + yy) + zz;
    *r2out = r2;
    return r2 < rr;
}

/* counts[i] = number of j > i with (i,j) in range.  O(N^2). */
void orc_nl_row_counts(int64_t n, const double *pos, const double box[3],
                       double rlist, int64_t *counts)
{
    const double rr = rlist * rlist;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = 0;
        int s[3];
        double d[3], r2;
        for (int64_t j = i + 1; j < n; ++j)
            c += orc_pair(pos + 3 * i, pos + 3 * j, box, rr, s, d, &r2);
        counts[i] = c;
    }
}

/* Fills the canonical list: unique pairs i<j sorted by (i,j), shift int8[3]
 * such that r_j + shift*box - r_i is the in-range vector.  offsets[i] is the
 * exclusive prefix sum of orc_nl_row_counts. */
void orc_nl_fill(int64_t n, const double *pos, const double box[3],
                 double rlist, const int64_t *offsets, int32_t *pi,
                 int32_t *pj, int8_t *shift)
{
    const double rr = rlist * rlist;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        int64_t o = offsets[i];
        int s[3];
        double d[3], r2;
        for (int64_t j = i + 1; j < n; ++j) {
            if (orc_pair(pos + 3 * i, pos + 3 * j, box, rr, s, d, &r2)) {
                pi[o] = (int32_t)i;
                pj[o] = (int32_t)j;
                shift[3 * o + 0] = (int8_t)s[0];
                shift[3 * o + 1] = (int8_t)s[1];
                shift[3 * o + 2] = (int8_t)s[2];
                ++o;
            }
        }
    }
}

/* Rows i0 <= i < i1 of the canonical list (j > i, ascending j) in ONE O((i1-i0) N) pass with
 * a fixed capacity per row: row i's entries go to pj[(i-i0)*cap ...], shift likewise, and
 * counts[i-i0] is the number found (entries beyond cap are counted, not written).  The same
 * predicate as orc_nl_fill; lets a test walk a large system chunk by chunk in bounded memory. */
void orc_nl_rows_upper(int64_t n, const double *pos, const double box[3],
                       double rlist, int64_t i0, int64_t i1, int64_t cap,
                       int64_t *counts, int32_t *pj, int8_t *shift)
{
    const double rr = rlist * rlist;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = i0; i < i1; ++i) {
        int64_t c = 0;
        int s[3];
        double d[3], r2;
        int32_t *oj = pj + (i - i0) * cap;
        int8_t *os = shift + 3 * (i - i0) * cap;
        for (int64_t j = i + 1; j < n; ++j) {
            if (orc_pair(pos + 3 * i, pos + 3 * j, box, rr, s, d, &r2)) {
                if (c < cap) {
                    oj[c] = (int32_t)j;
                    os[3 * c + 0] = (int8_t)s[0];
                    os[3 * c + 1] = (int8_t)s[1];
                    os[3 * c + 2] = (int8_t)s[2];
                }
                ++c;
            }
        }
        counts[i - i0] = c;
    }
}

/* All neighbours j != i of ONE atom i (directed row), ascending j, with the
 * shift for the ordered pair (i,j).  Returns the number found (writes at most
 * cap of them).  O(N) -- used to check sampled rows at sizes where the full
 * O(N^2) search is too slow. */
int64_t orc_nl_row(int64_t n, const double *pos, const double box[3],
                   double rlist, int64_t i, int64_t cap, int32_t *out_j,
                   int8_t *out_shift)
{
    const double rr = rlist * rlist;
    int64_t c = 0;
    int s[3];
    double d[3], r2;
    for (int64_t j = 0; j < n; ++j) {
        if (j == i) continue;
        if (orc_pair(pos + 3 * i, pos + 3 * j, box, rr, s, d, &r2)) {
            if (c < cap) {
                out_j[c] = (int32_t)j;
                out_shift[3 * c + 0] = (int8_t)s[0];
                out_shift[3 * c + 1] = (int8_t)s[1];
                out_shift[3 * c + 2] = (int8_t)s[2];
            }
            ++c;
        }
    }
    return c;
}

/* ------------------------------------------------------------------------ */
/* c-RS: real-space part, Eq. 3 restricted to r < rc with the  */
/* minimum image (one image per pair; needs rc < L/2).         */
/*   t = erfc(alpha r)/r                     phi_i += q_j t                  */
/*   g = (t + (2 alpha/sqrt(pi)) exp(-alpha^2 r^2)) / r^2                    */
/*   F_i += q_i q_j g (r_i - r_j - s L)      (F = -dE/dr)                    */
/* ------------------------------------------------------------------------ */
static void orc_realspace_one(int64_t n, const double *pos, const double *q,
                              const double box[3], double rc, double alpha,
                              int64_t i, double *phi_i, double *F_i)
{
    const double rr = rc * rc;
    const double c2 = 2.0 * alpha / sqrt(ORC_PI);
    double p = 0.0, fx = 0.0, fy = 0.0, fz = 0.0;
    int s[3];
    double d[3], r2;
    for (int64_t j = 0; j < n; ++j) {
        if (j == i) continue;
        if (!orc_pair(pos + 3 * i, pos + 3 * j, box, rr, s, d, &r2)) continue;
        double r = sqrt(r2);
        double t = erfc(alpha * r) / r;
        double g = (t + c2 * exp(-alpha * alpha * r2)) / r2;
        p += q[j] * t;
        double qq = q[i] * q[j] * g;
        fx += qq * (-d[0]);
        fy += qq * (-d[1]);
        fz += qq * (-d[2]);
    }
    *phi_i = p;
    F_i[0] = fx;
    F_i[1] = fy;
    F_i[2] = fz;
}

void orc_realspace(int64_t n, const double *pos, const double *q,
                   const double box[3], double rc, double alpha, double *phi,
                   double *F)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i)
        orc_realspace_one(n, pos, q, box, rc, alpha, i, phi + i, F + 3 * i);
}

void orc_realspace_rows(int64_t n, const double *pos, const double *q,
                        const double box[3], double rc, double alpha,
                        int64_t nrows, const int64_t *rows, double *phi,
                        double *F)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t k = 0; k < nrows; ++k)
        orc_realspace_one(n, pos, q, box, rc, alpha, rows[k], phi + k,
                          F + 3 * k);
}

/* ------------------------------------------------------------------------ */
/* c-EW: direct (regular) Ewald summation, Eqs. 2-5.        */
/* Real space: all images n with |n_d| <= nimg[d], all pairs including the   */
/* self images (i=j, n!=0) (reading G8), r < rcut_real.                      */
/* Reciprocal: k = 2 pi m / L for all integer m != 0 with |m_d| <= mmax[d];  */
/*   S(k) = sum_j q_j e^{i k.r_j};  E_rec = (2 pi/V) sum_k v_k |S|^2,        */
/*   v_k = exp(-k^2/4 alpha^2)/k^2  (Eq. 4; reading G1)                      */
/*   phi_i^rec = (4 pi/V) sum_k v_k [cos(k.r_i) Re S + sin(k.r_i) Im S]      */
/*   dE/dr_i   = (4 pi/V) sum_k v_k k q_i [cos(k.r_i) Im S - sin(k.r_i) Re S]*/
/*   (the gradient of Eq. 6; reading G2).   Self: phi_i -= 2 alpha/sqrt(pi) q_i. */
/* background != 0 adds the neutralising-background term -pi Q/(V alpha^2)   */
/* to phi (needed only for checks on non-neutral q; reading G11).            */
/* Outputs: phi[n], F[3n] (= -dE/dr), *E = (1/2) sum q phi.                  */
/* ------------------------------------------------------------------------ */
void orc_ewald_direct(int64_t n, const double *pos, const double *q,
                      const double box[3], double alpha, double rcut_real,
                      const int nimg[3], const int mmax[3], int background,
                      double *phi, double *F, double *E)
{
    const double V = box[0] * box[1] * box[2];
    const double c2 = 2.0 * alpha / sqrt(ORC_PI);
    const double rr = rcut_real * rcut_real;
    for (int64_t i = 0; i < n; ++i) {
        phi[i] = 0.0;
        F[3 * i] = F[3 * i + 1] = F[3 * i + 2] = 0.0;
    }
    /* real space */
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < n; ++i) {
        double p = 0.0, f[3] = {0.0, 0.0, 0.0};
        for (int64_t j = 0; j < n; ++j)
            for (int a = -nimg[0]; a <= nimg[0]; ++a)
                for (int b = -nimg[1]; b <= nimg[1]; ++b)
                    for (int c = -nimg[2]; c <= nimg[2]; ++c) {
                        if (j == i && a == 0 && b == 0 && c == 0) continue;
                        double dx = pos[3 * i] - pos[3 * j] - a * box[0];
                        double dy = pos[3 * i + 1] - pos[3 * j + 1] - b * box[1];
                        double dz = pos[3 * i + 2] - pos[3 * j + 2] - c * box[2];
                        double r2 = dx * dx + dy * dy + dz * dz;
                        if (!(r2 < rr)) continue;
                        double r = sqrt(r2);
                        double t = erfc(alpha * r) / r;
                        double g = (t + c2 * exp(-alpha * alpha * r2)) / r2;
                        p += q[j] * t;
                        f[0] += q[i] * q[j] * g * dx;
                        f[1] += q[i] * q[j] * g * dy;
                        f[2] += q[i] * q[j] * g * dz;
                    }
        phi[i] += p;
        F[3 * i] += f[0];
        F[3 * i + 1] += f[1];
        F[3 * i + 2] += f[2];
    }
    /* reciprocal space: one k-vector at a time */
    const int64_t nmx = 2 * mmax[0] + 1, nmy = 2 * mmax[1] + 1,
                  nmz = 2 * mmax[2] + 1;
    const int64_t nk = nmx * nmy * nmz;
    int nth = orc_num_threads();
    double *acc = (double *)calloc((size_t)nth * 4 * n, sizeof(double));
#pragma omp parallel
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        double *ap = acc + (size_t)tid * 4 * n;
        double *cs = (double *)malloc(2 * n * sizeof(double));
#pragma omp for schedule(dynamic, 4)
        for (int64_t ik = 0; ik < nk; ++ik) {
            int mx = (int)(ik / (nmy * nmz)) - mmax[0];
            int my = (int)((ik / nmz) % nmy) - mmax[1];
            int mz = (int)(ik % nmz) - mmax[2];
            if (mx == 0 && my == 0 && mz == 0) continue;
            double kx = 2.0 * ORC_PI * mx / box[0];
            double ky = 2.0 * ORC_PI * my / box[1];
            double kz = 2.0 * ORC_PI * mz / box[2];
            double k2 = kx * kx + ky * ky + kz * kz;
            double v = exp(-k2 / (4.0 * alpha * alpha)) / k2;
            if (v == 0.0) continue;
            double sre = 0.0, sim = 0.0;
            for (int64_t j = 0; j < n; ++j) {
                double ph = kx * pos[3 * j] + ky * pos[3 * j + 1] +
                            kz * pos[3 * j + 2];
                cs[2 * j] = cos(ph);
                cs[2 * j + 1] = sin(ph);
                sre += q[j] * cs[2 * j];
                sim += q[j] * cs[2 * j + 1];
            }
            double pref = 4.0 * ORC_PI / V * v;
            for (int64_t i = 0; i < n; ++i) {
                double c = cs[2 * i], s = cs[2 * i + 1];
                ap[4 * i] += pref * (c * sre + s * sim);
                double dEd = pref * q[i] * (c * sim - s * sre);
                ap[4 * i + 1] -= dEd * kx;
                ap[4 * i + 2] -= dEd * ky;
                ap[4 * i + 3] -= dEd * kz;
            }
        }
        free(cs);
    }
    double Q = 0.0;
    for (int64_t i = 0; i < n; ++i) Q += q[i];
    double e = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        for (int t = 0; t < nth; ++t) {
            const double *ap = acc + (size_t)t * 4 * n;
            phi[i] += ap[4 * i];
            F[3 * i] += ap[4 * i + 1];
            F[3 * i + 1] += ap[4 * i + 2];
            F[3 * i + 2] += ap[4 * i + 3];
        }
        phi[i] -= c2 * q[i];
        if (background) phi[i] -= ORC_PI * Q / (V * alpha * alpha);
        e += 0.5 * q[i] * phi[i];
    }
    free(acc);
    *E = e;
}

/* ------------------------------------------------------------------------ */
/* Cardinal B-spline M_n(u), support (0,n) (the "cardinal B-spline           */
/* interpolation" of Alg. 2 step 1; recursion as in        */
/* DESIGN.md R-PME):                                                         */
/*   M_2(u) = 1-|u-1| on [0,2];                                              */
/*   M_n(u) = [u M_{n-1}(u) + (n-u) M_{n-1}(u-1)]/(n-1)                      */
/*   M_n'(u) = M_{n-1}(u) - M_{n-1}(u-1)                                     */
/* ------------------------------------------------------------------------ */
double orc_bspline(int n, double u)
{
    if (n == 2) {
        if (u < 0.0 || u > 2.0) return 0.0;
        return 1.0 - fabs(u - 1.0);
    }
    return (u * orc_bspline(n - 1, u) + (n - u) * orc_bspline(n - 1, u - 1.0)) /
           (n - 1);
}

double orc_bspline_deriv(int n, double u)
{
    return orc_bspline(n - 1, u) - orc_bspline(n - 1, u - 1.0);
}

/* Step 1 bookkeeping for one atom and one axis:
 *   u = frac(x/L) K in [0,K);  f = floor(u);  w = u - f;
 *   theta[j] = M_p(w+j), dtheta[j] = M_p'(w+j) on grid index (f-j) mod K. */
static void orc_axis_weights(double x, double L, int K, int p, int *idx,
                             double *theta, double *dtheta)
{
    double s = x / L;
    s = s - floor(s);
    double u = s * K;
    int f = (int)floor(u);
    if (f >= K) { /* s rounded up to 1.0 */
        f -= K;
        u -= K;
    }
    double w = u - f;
    for (int j = 0; j < p; ++j) {
        int g = (f - j) % K;
        if (g < 0) g += K;
        idx[j] = g;
        theta[j] = orc_bspline(p, w + j);
        dtheta[j] = orc_bspline_deriv(p, w + j);
    }
}

/* Alg. 2 step 1: Q(k) += q_i theta_x theta_y theta_z.
 * Q is [K0][K1][K2] row-major, zeroed here.  Serial: summation order fixed. */
void orc_pme_spread(int64_t n, const double *pos, const double *q,
                    const double box[3], const int K[3], int p, double *Q)
{
    int ix[16], iy[16], iz[16];
    double tx[16], ty[16], tz[16], dx[16], dy[16], dz[16];
    memset(Q, 0, sizeof(double) * (size_t)K[0] * K[1] * K[2]);
    for (int64_t i = 0; i < n; ++i) {
        orc_axis_weights(pos[3 * i], box[0], K[0], p, ix, tx, dx);
        orc_axis_weights(pos[3 * i + 1], box[1], K[1], p, iy, ty, dy);
        orc_axis_weights(pos[3 * i + 2], box[2], K[2], p, iz, tz, dz);
        for (int a = 0; a < p; ++a)
            for (int b = 0; b < p; ++b)
                for (int c = 0; c < p; ++c)
                    Q[((size_t)ix[a] * K[1] + iy[b]) * K[2] + iz[c]] +=
                        q[i] * tx[a] * ty[b] * tz[c];
    }
}

/* Alg. 2 steps 2 and 4: unnormalised 3-D DFT of a complex
 * array z[K0][K1][K2] (interleaved re,im), in place, as three sweeps of naive
 * O(K^2) line DFTs:  out[m] = sum_k in[k] exp(sign 2 pi i m k / K).         */
static void orc_dft_axis(double *z, const int K[3], int axis, int sign)
{
    const int Ka = K[axis];
    /* a line along `axis` starts at element (o * Ka * ninner + r) and steps by
     * `stride` = ninner elements; o < nouter, r < ninner */
    int64_t stride, nouter, ninner;
    if (axis == 2) { nouter = (int64_t)K[0] * K[1]; ninner = 1; }
    else if (axis == 1) { nouter = K[0]; ninner = K[2]; }
    else { nouter = 1; ninner = (int64_t)K[1] * K[2]; }
    stride = ninner;
    double *tw = (double *)malloc(sizeof(double) * 2 * Ka);
    for (int t = 0; t < Ka; ++t) {
        tw[2 * t] = cos(2.0 * ORC_PI * t / Ka);
        tw[2 * t + 1] = sign * sin(2.0 * ORC_PI * t / Ka);
    }
    const int64_t nlines = nouter * ninner;
#pragma omp parallel
    {
        double *in = (double *)malloc(sizeof(double) * 2 * Ka);
#pragma omp for schedule(static)
        for (int64_t l = 0; l < nlines; ++l) {
            int64_t o = l / ninner, r = l % ninner;
            double *base = z + 2 * (o * Ka * ninner + r);
            for (int k = 0; k < Ka; ++k) {
                in[2 * k] = base[2 * k * stride];
                in[2 * k + 1] = base[2 * k * stride + 1];
            }
            for (int m = 0; m < Ka; ++m) {
                double re = 0.0, im = 0.0;
                for (int k = 0; k < Ka; ++k) {
                    int t = (int)(((int64_t)m * k) % Ka);
                    re += in[2 * k] * tw[2 * t] - in[2 * k + 1] * tw[2 * t + 1];
                    im += in[2 * k] * tw[2 * t + 1] + in[2 * k + 1] * tw[2 * t];
                }
                base[2 * m * stride] = re;
                base[2 * m * stride + 1] = im;
            }
        }
        free(in);
    }
    free(tw);
}

void orc_dft3(double *z, const int K[3], int sign)
{
    orc_dft_axis(z, K, 2, sign);
    orc_dft_axis(z, K, 1, sign);
    orc_dft_axis(z, K, 0, sign);
}

/* |b(m)|^2 = 1 / | sum_{k=0}^{p-2} M_p(k+1) e^{2 pi i m k/K} |^2  (DESIGN.md R-PME) */
static double orc_bmod2(int m, int K, int p)
{
    /* odd p, m = K/2: the sum below is exactly zero (M_p(k+1) is symmetric in k about (p-2)/2 and the signs
     * alternate), the order-p exponential spline cannot carry the Nyquist frequency.  The paper is silent on odd
     * orders; reading G19: that plane is left out, |b|^2 := 0, hence G = 0 there. */
    if ((p & 1) && 2 * m == K) return 0.0;
    double re = 0.0, im = 0.0;
    for (int k = 0; k <= p - 2; ++k) {
        double a = 2.0 * ORC_PI * (double)m * (double)k / (double)K;
        double M = orc_bspline(p, (double)(k + 1));
        re += M * cos(a);
        im += M * sin(a);
    }
    return 1.0 / (re * re + im * im);
}

/* Influence function G(m) = B(m) C(m), G(0) = 0:
 *   B = prod_d |b_d(m_d)|^2,  C = exp(-pi^2 mt^2/alpha^2)/(pi V mt^2),
 *   mt_d = m'_d / L_d,  m' = m if m <= K/2 else m-K.
 * Equivalent to the (4 pi/k^2) exp(-k^2/4 alpha^2)/(2V)... factor of Eq. 4
 * with k = 2 pi mt, times the B-spline deconvolution. */
void orc_pme_influence_table(const double box[3], const int K[3], int p,
                             double alpha, double *G)
{
    const double V = box[0] * box[1] * box[2];
    double *b[3];
    for (int d = 0; d < 3; ++d) {
        b[d] = (double *)malloc(sizeof(double) * K[d]);
        for (int m = 0; m < K[d]; ++m) b[d][m] = orc_bmod2(m, K[d], p);
    }
    for (int m0 = 0; m0 < K[0]; ++m0)
        for (int m1 = 0; m1 < K[1]; ++m1)
            for (int m2 = 0; m2 < K[2]; ++m2) {
                size_t o = ((size_t)m0 * K[1] + m1) * K[2] + m2;
                if (m0 == 0 && m1 == 0 && m2 == 0) { G[o] = 0.0; continue; }
                double a0 = (m0 <= K[0] / 2 ? m0 : m0 - K[0]) / box[0];
                double a1 = (m1 <= K[1] / 2 ? m1 : m1 - K[1]) / box[1];
                double a2 = (m2 <= K[2] / 2 ? m2 : m2 - K[2]) / box[2];
                double mt2 = a0 * a0 + a1 * a1 + a2 * a2;
                double C = exp(-ORC_PI * ORC_PI * mt2 / (alpha * alpha)) /
                           (ORC_PI * V * mt2);
                G[o] = b[0][m0] * b[1][m1] * b[2][m2] * C;
            }
    for (int d = 0; d < 3; ++d) free(b[d]);
}

/* Alg. 2 step 5: phi_i = sum theta theta theta Phi;
 * F_i,x = -q_i (K_x/L_x) sum theta'_x theta_y theta_z Phi (cyclic). */
void orc_pme_gather(int64_t n, const double *pos, const double *q,
                    const double box[3], const int K[3], int p,
                    const double *Phi, double *phi, double *F)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int ix[16], iy[16], iz[16];
        double tx[16], ty[16], tz[16], dx[16], dy[16], dz[16];
        orc_axis_weights(pos[3 * i], box[0], K[0], p, ix, tx, dx);
        orc_axis_weights(pos[3 * i + 1], box[1], K[1], p, iy, ty, dy);
        orc_axis_weights(pos[3 * i + 2], box[2], K[2], p, iz, tz, dz);
        double s = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
        for (int a = 0; a < p; ++a)
            for (int b = 0; b < p; ++b)
                for (int c = 0; c < p; ++c) {
                    double P = Phi[((size_t)ix[a] * K[1] + iy[b]) * K[2] + iz[c]];
                    s += tx[a] * ty[b] * tz[c] * P;
                    gx += dx[a] * ty[b] * tz[c] * P;
                    gy += tx[a] * dy[b] * tz[c] * P;
                    gz += tx[a] * ty[b] * dz[c] * P;
                }
        phi[i] = s;
        F[3 * i] = -q[i] * (K[0] / box[0]) * gx;
        F[3 * i + 1] = -q[i] * (K[1] / box[1]) * gy;
        F[3 * i + 2] = -q[i] * (K[2] / box[2]) * gz;
    }
}

/* Alg. 2, all five steps.  Outputs phi_rec[n], F_rec[3n],
 * *E_rec = (1/2) sum_m G |Qhat|^2 over the full spectrum.  Optional outputs
 * (may be NULL): Qgrid[K0 K1 K2] = the charge grid after step 1, Phigrid =
 * the potential grid after step 4 (unnormalised inverse: no 1/K^3). */
void orc_pme_recip(int64_t n, const double *pos, const double *q,
                   const double box[3], const int K[3], int p, double alpha,
                   double *phi, double *F, double *E_rec, double *Qgrid,
                   double *Phigrid)
{
    const size_t G3 = (size_t)K[0] * K[1] * K[2];
    double *Q = (double *)malloc(sizeof(double) * G3);
    double *z = (double *)malloc(sizeof(double) * 2 * G3);
    double *G = (double *)malloc(sizeof(double) * G3);
    orc_pme_spread(n, pos, q, box, K, p, Q);                 /* step 1 */
    if (Qgrid) memcpy(Qgrid, Q, sizeof(double) * G3);
    for (size_t o = 0; o < G3; ++o) { z[2 * o] = Q[o]; z[2 * o + 1] = 0.0; }
    orc_dft3(z, K, -1);                                      /* step 2 */
    orc_pme_influence_table(box, K, p, alpha, G);            /* step 3 */
    double e = 0.0;
    for (size_t o = 0; o < G3; ++o) {
        e += 0.5 * G[o] * (z[2 * o] * z[2 * o] + z[2 * o + 1] * z[2 * o + 1]);
        z[2 * o] *= G[o];
        z[2 * o + 1] *= G[o];
    }
    *E_rec = e;
    orc_dft3(z, K, +1);                                      /* step 4 */
    for (size_t o = 0; o < G3; ++o) Q[o] = z[2 * o];
    if (Phigrid) memcpy(Phigrid, Q, sizeof(double) * G3);
    orc_pme_gather(n, pos, q, box, K, p, Q, phi, F);         /* step 5 */
    free(Q);
    free(z);
    free(G);
}
