"""fp64 CPU oracle for the periodic Coulomb path of arxiv 2503.21176.

TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT PATH.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It shares no code with paper_2503_21176_b200/ and
neither imports the other.

The arithmetic lives in sqeq_oracle.c (plain C, fp64, OpenMP over independent
outer iterations); this module only marshals numpy arrays into it and writes
out, in numpy, the few dense linear-algebra definitions (QEq KKT system,
Eq. 18; the shadow-MD closed form, Eq. 22).  Inputs may be fp32 arrays (the
very arrays the GPU receives); they are promoted to fp64 exactly and
everything after that is fp64.

Citations: PAPER.md:N = line N of /root/reference/PAPER.md.
Pins (tests/test_oracle_*.py): rock-salt / CsCl / zincblende Madelung
constants, the cubic self-image constant xi, alpha-independence, finite
differences, PME grid-shift invariance and operator symmetry, numpy.fft,
scipy B-splines, scipy periodic cKDTree, brute-force multi-image sums.
Functions whose parity is unpinned: shadow_md_step / shadow_md_init (the n(t)
integrator's constants and history start are not given by the paper -- DESIGN.md
R-MD); their ingredients (Eq. 22, shadow forces = -grad U, Eq. 24's J, GMRES) are pinned.
"""
import ctypes
import math
import os

import numpy as np

from . import build as _build

KE_EV_A = 14.3996454784255  # e^2/(4 pi eps0) in eV*Angstrom (DESIGN.md R-units)

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        c_dp = ctypes.POINTER(ctypes.c_double)
        c_ip = ctypes.POINTER(ctypes.c_int)
        i64 = ctypes.c_int64
        L.orc_num_threads.restype = ctypes.c_int
        L.orc_nl_row_counts.argtypes = [i64, c_dp, c_dp, ctypes.c_double, ctypes.c_void_p]
        L.orc_nl_fill.argtypes = [i64, c_dp, c_dp, ctypes.c_double, ctypes.c_void_p,
                                  ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.orc_nl_row.argtypes = [i64, c_dp, c_dp, ctypes.c_double, i64, i64,
                                 ctypes.c_void_p, ctypes.c_void_p]
        L.orc_nl_row.restype = i64
        L.orc_nl_rows_upper.argtypes = [i64, c_dp, c_dp, ctypes.c_double, i64, i64, i64,
                                        ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.orc_realspace.argtypes = [i64, c_dp, c_dp, c_dp, ctypes.c_double,
                                    ctypes.c_double, c_dp, c_dp]
        L.orc_realspace_rows.argtypes = [i64, c_dp, c_dp, c_dp, ctypes.c_double,
                                         ctypes.c_double, i64, ctypes.c_void_p, c_dp, c_dp]
        L.orc_ewald_direct.argtypes = [i64, c_dp, c_dp, c_dp, ctypes.c_double,
                                       ctypes.c_double, c_ip, c_ip, ctypes.c_int,
                                       c_dp, c_dp, c_dp]
        L.orc_bspline.argtypes = [ctypes.c_int, ctypes.c_double]
        L.orc_bspline.restype = ctypes.c_double
        L.orc_bspline_deriv.argtypes = [ctypes.c_int, ctypes.c_double]
        L.orc_bspline_deriv.restype = ctypes.c_double
        L.orc_pme_spread.argtypes = [i64, c_dp, c_dp, c_dp, c_ip, ctypes.c_int, c_dp]
        L.orc_dft3.argtypes = [c_dp, c_ip, ctypes.c_int]
        L.orc_pme_influence_table.argtypes = [c_dp, c_ip, ctypes.c_int, ctypes.c_double, c_dp]
        L.orc_pme_gather.argtypes = [i64, c_dp, c_dp, c_dp, c_ip, ctypes.c_int, c_dp, c_dp, c_dp]
        L.orc_pme_recip.argtypes = [i64, c_dp, c_dp, c_dp, c_ip, ctypes.c_int,
                                    ctypes.c_double, c_dp, c_dp, c_dp, c_dp, c_dp]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a), dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _box(box):
    b = _f64(box).reshape(-1)
    if b.size == 1:
        b = np.repeat(b, 3)
    assert b.size == 3
    return np.ascontiguousarray(b)


# --------------------------------------------------------------------------
# c-NL  neighbour list = the plain O(N^2) definition (Alg. 1)
# --------------------------------------------------------------------------
def neighbour_list(pos, box, rlist):
    """Unique pairs i<j sorted by (i,j) with int8 shift s.t. r_j + s*L - r_i is in range."""
    pos = _f64(pos, (-1, 3))
    box = _box(box)
    n = pos.shape[0]
    counts = np.zeros(n, dtype=np.int64)
    lib().orc_nl_row_counts(n, _dp(pos), _dp(box), float(rlist), counts.ctypes.data)
    offsets = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=offsets[1:])
    tot = int(offsets[-1])
    pi = np.empty(tot, dtype=np.int32)
    pj = np.empty(tot, dtype=np.int32)
    sh = np.empty((tot, 3), dtype=np.int8)
    lib().orc_nl_fill(n, _dp(pos), _dp(box), float(rlist), offsets.ctypes.data,
                      pi.ctypes.data, pj.ctypes.data, sh.ctypes.data)
    return pi, pj, sh


def neighbour_rows_upper(pos, box, rlist, i0, i1, cap=1024):
    """Rows i0 <= i < i1 of the canonical list (j > i) in one pass: (i, j, shift) arrays sorted by
    (i, j), exactly the slice of neighbour_list() with i0 <= i < i1."""
    pos = _f64(pos, (-1, 3))
    box = _box(box)
    n = pos.shape[0]
    while True:
        m = int(i1 - i0)
        counts = np.zeros(m, dtype=np.int64)
        pj = np.empty((m, cap), dtype=np.int32)
        sh = np.empty((m, cap, 3), dtype=np.int8)
        lib().orc_nl_rows_upper(n, _dp(pos), _dp(box), float(rlist), int(i0), int(i1), int(cap),
                                counts.ctypes.data, pj.ctypes.data, sh.ctypes.data)
        if counts.max(initial=0) <= cap:
            break
        cap = int(counts.max())
    mask = np.arange(cap)[None, :] < counts[:, None]
    oi = np.repeat(np.arange(i0, i1, dtype=np.int32), counts)
    return oi, pj[mask], sh[mask]


def neighbour_row(pos, box, rlist, i, cap=4096):
    """All neighbours j != i of atom i (ascending j) and the shift of the ordered pair (i,j)."""
    pos = _f64(pos, (-1, 3))
    box = _box(box)
    n = pos.shape[0]
    while True:
        oj = np.empty(cap, dtype=np.int32)
        os_ = np.empty((cap, 3), dtype=np.int8)
        c = int(lib().orc_nl_row(n, _dp(pos), _dp(box), float(rlist), int(i), cap,
                                 oj.ctypes.data, os_.ctypes.data))
        if c <= cap:
            return oj[:c].copy(), os_[:c].copy()
        cap = c


# --------------------------------------------------------------------------
# c-RS  real-space erfc sum, Eq. 3, r < rc, minimum image
# --------------------------------------------------------------------------
def realspace(pos, q, box, rc, alpha):
    pos = _f64(pos, (-1, 3)); q = _f64(q); box = _box(box)
    n = pos.shape[0]
    phi = np.zeros(n); F = np.zeros((n, 3))
    lib().orc_realspace(n, _dp(pos), _dp(q), _dp(box), float(rc), float(alpha), _dp(phi), _dp(F))
    return phi, F


def realspace_rows(pos, q, box, rc, alpha, rows):
    pos = _f64(pos, (-1, 3)); q = _f64(q); box = _box(box)
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    n = pos.shape[0]
    phi = np.zeros(rows.size); F = np.zeros((rows.size, 3))
    lib().orc_realspace_rows(n, _dp(pos), _dp(q), _dp(box), float(rc), float(alpha),
                             rows.size, rows.ctypes.data, _dp(phi), _dp(F))
    return phi, F


# --------------------------------------------------------------------------
# c-EW  direct Ewald, Eqs. 2-5 -- pins PME, not a parity target
# --------------------------------------------------------------------------
def ewald_direct(pos, q, box, alpha, tol=1e-16, background=False):
    """Converged regular Ewald sum: phi, F (= -dE/dr), E = 1/2 sum q phi.

    The real-space sum runs over all images with erfc(alpha r) above `tol`, the
    reciprocal sum over all k with exp(-k^2/4 alpha^2) above `tol`.
    """
    pos = _f64(pos, (-1, 3)); q = _f64(q); box = _box(box)
    n = pos.shape[0]
    x = math.sqrt(-math.log(tol))          # erfc(x) < exp(-x^2) = tol
    rcut = x / alpha
    kmax = 2.0 * alpha * x                 # exp(-k^2/4a^2) = tol
    nimg = np.array([int(math.ceil(rcut / L)) for L in box], dtype=np.intc)
    mmax = np.array([int(math.ceil(kmax * L / (2 * math.pi))) for L in box], dtype=np.intc)
    phi = np.zeros(n); F = np.zeros((n, 3)); E = np.zeros(1)
    lib().orc_ewald_direct(n, _dp(pos), _dp(q), _dp(box), float(alpha), float(rcut),
                           _ip(nimg), _ip(mmax), int(bool(background)), _dp(phi), _dp(F), _dp(E))
    return phi, F, float(E[0])


def ewald_truncated(pos, q, box, rc, alpha, kmax):
    """Regular Ewald with the cutoffs of a production run: real space over minimum-image pairs
    with r < rc (rc < L/2), reciprocal space over all m != 0 with |m_d| <= kmax[d], self term.  The same routine as
    ewald_direct with those cutoffs given instead of derived from a tolerance.  Returns phi, F, E."""
    pos = _f64(pos, (-1, 3)); q = _f64(q); box = _box(box)
    n = pos.shape[0]
    # the C routine visits images -1, 0, +1 of the positions it is given: hand it the positions wrapped into the box
    # (nothing changes physically: the real-space sum is over images, the phases are periodic)
    pos = pos - np.floor(pos / box) * box
    nimg = np.ones(3, dtype=np.intc)
    mmax = np.ascontiguousarray(np.asarray(kmax, dtype=np.intc).reshape(3))
    phi = np.zeros(n); F = np.zeros((n, 3)); E = np.zeros(1)
    lib().orc_ewald_direct(n, _dp(pos), _dp(q), _dp(box), float(alpha), float(rc), _ip(nimg), _ip(mmax), 0,
                           _dp(phi), _dp(F), _dp(E))
    return phi, F, float(E[0])


# --------------------------------------------------------------------------
# c-PME  smooth PME, Alg. 2
# --------------------------------------------------------------------------
def bspline(n, u):
    return float(lib().orc_bspline(int(n), float(u)))


def bspline_deriv(n, u):
    return float(lib().orc_bspline_deriv(int(n), float(u)))


def _grid(grid):
    g = np.asarray(grid, dtype=np.intc).reshape(-1)
    if g.size == 1:
        g = np.repeat(g, 3)
    return np.ascontiguousarray(g, dtype=np.intc)


def pme_spread(pos, q, box, grid, order):
    pos = _f64(pos, (-1, 3)); q = _f64(q); box = _box(box); K = _grid(grid)
    Q = np.zeros(tuple(int(k) for k in K))
    lib().orc_pme_spread(pos.shape[0], _dp(pos), _dp(q), _dp(box), _ip(K), int(order), _dp(Q))
    return Q


def dft3(z, sign):
    """Unnormalised 3-D DFT, out[m] = sum_k z[k] exp(sign 2 pi i m.k/K), naive line DFTs."""
    z = np.ascontiguousarray(z, dtype=np.complex128).copy()
    K = np.array(z.shape, dtype=np.intc)
    lib().orc_dft3(z.view(np.float64).ctypes.data_as(ctypes.POINTER(ctypes.c_double)), _ip(K), int(sign))
    return z


def pme_influence(box, grid, order, alpha):
    box = _box(box); K = _grid(grid)
    G = np.zeros(tuple(int(k) for k in K))
    lib().orc_pme_influence_table(_dp(box), _ip(K), int(order), float(alpha), _dp(G))
    return G


def pme_gather(pos, q, box, grid, order, Phi):
    """Alg. 2 step 5 alone: phi_i = sum W Phi, F_i = -q_i (K/L) sum dW Phi on a given grid Phi."""
    pos = _f64(pos, (-1, 3)); q = _f64(q); box = _box(box); K = _grid(grid)
    Phi = np.ascontiguousarray(Phi, dtype=np.float64)
    n = pos.shape[0]
    phi = np.zeros(n); F = np.zeros((n, 3))
    lib().orc_pme_gather(n, _dp(pos), _dp(q), _dp(box), _ip(K), int(order), _dp(Phi), _dp(phi), _dp(F))
    return phi, F


def pme_recip(pos, q, box, grid, order, alpha, return_grids=False):
    """Alg. 2 steps 1-5: phi_rec, F_rec, E_rec (and optionally the Q and Phi grids)."""
    pos = _f64(pos, (-1, 3)); q = _f64(q); box = _box(box); K = _grid(grid)
    n = pos.shape[0]
    phi = np.zeros(n); F = np.zeros((n, 3)); E = np.zeros(1)
    shape = tuple(int(k) for k in K)
    if return_grids:
        Qg = np.zeros(shape); Pg = np.zeros(shape)
        lib().orc_pme_recip(n, _dp(pos), _dp(q), _dp(box), _ip(K), int(order), float(alpha),
                            _dp(phi), _dp(F), _dp(E), _dp(Qg), _dp(Pg))
        return phi, F, float(E[0]), Qg, Pg
    lib().orc_pme_recip(n, _dp(pos), _dp(q), _dp(box), _ip(K), int(order), float(alpha),
                        _dp(phi), _dp(F), _dp(E), None, None)
    return phi, F, float(E[0])


def self_potential(q, alpha):
    """phi_i^self = -(2 alpha/sqrt(pi)) q_i, from E_self of Eq. 5."""
    return -(2.0 * alpha / math.sqrt(math.pi)) * _f64(q)


def coulomb_pme(pos, q, box, rc, alpha, grid, order, rows=None):
    """Total PME Coulomb evaluation (Eq. 2): real(r<rc) + reciprocal + self.

    Returns phi (dE/dq), F (-dE/dr), E = 1/2 sum q phi, and a dict of the parts.
    With `rows` given, the O(N^2) real-space part is evaluated only for those
    atoms and phi, F are returned for those rows only (E is then None).
    """
    q64 = _f64(q)
    p_rec, F_rec, E_rec = pme_recip(pos, q, box, grid, order, alpha)
    p_self = self_potential(q, alpha)
    if rows is None:
        p_real, F_real = realspace(pos, q, box, rc, alpha)
        phi = p_real + p_rec + p_self
        F = F_real + F_rec
        E = 0.5 * float(np.dot(q64, phi))
        parts = dict(phi_real=p_real, F_real=F_real, phi_rec=p_rec, F_rec=F_rec,
                     phi_self=p_self, E_rec=E_rec,
                     E_real=0.5 * float(np.dot(q64, p_real)),
                     E_self=0.5 * float(np.dot(q64, p_self)))
        return phi, F, E, parts
    rows = np.asarray(rows, dtype=np.int64)
    p_real, F_real = realspace_rows(pos, q, box, rc, alpha, rows)
    phi = p_real + p_rec[rows] + p_self[rows]
    F = F_real + F_rec[rows]
    parts = dict(phi_real=p_real, F_real=F_real, phi_rec=p_rec[rows], F_rec=F_rec[rows],
                 E_rec=E_rec)
    return phi, F, None, parts


# --------------------------------------------------------------------------
# c-QEq  Eq. 18: [[C,1],[1^T,0]] [q;lambda] = [-chi; Qtot],
#        C v = J o v + ke * phi[v]   (sign reading G3)
# --------------------------------------------------------------------------
def coulomb_matrix_pme(pos, box, rc, alpha, grid, order):
    """Dense A with phi[v] = A v, column by column: A[:,j] = phi[e_j] (small N only)."""
    pos = _f64(pos, (-1, 3))
    n = pos.shape[0]
    A = np.zeros((n, n))
    e = np.zeros(n)
    for j in range(n):
        e[:] = 0.0
        e[j] = 1.0
        A[:, j] = coulomb_pme(pos, e, box, rc, alpha, grid, order)[0]
    return A


def qeq_kkt(A, chi, J, ke, qtot):
    """Assemble Eq. 18's (N+1)x(N+1) matrix and right-hand side."""
    n = A.shape[0]
    M = np.zeros((n + 1, n + 1))
    M[:n, :n] = ke * A + np.diag(_f64(J))
    M[:n, n] = 1.0
    M[n, :n] = 1.0
    b = np.concatenate([-_f64(chi), [float(qtot)]])
    return M, b


def qeq_dense_solve(A, chi, J, ke, qtot):
    """Solve Eq. 18 densely (LU with partial pivoting): returns q, lambda."""
    M, b = qeq_kkt(A, chi, J, ke, qtot)
    x = np.linalg.solve(M, b)
    return x[:-1], float(x[-1])


def qeq_residual(pos, box, rc, alpha, grid, order, chi, J, ke, qtot, q, lam):
    """True relative residual ||b - A x||/||b|| of Eq. 18 with the fp64 oracle mat-vec
    (the paper's convergence measure)."""
    q = _f64(q)
    phi = coulomb_pme(pos, q, box, rc, alpha, grid, order)[0]
    r_top = -_f64(chi) - (_f64(J) * q + ke * phi + lam)
    r_bot = float(qtot) - q.sum()
    bnorm = math.sqrt(float(np.dot(_f64(chi), _f64(chi))) + float(qtot) ** 2)
    return math.sqrt(float(np.dot(r_top, r_top)) + r_bot ** 2) / bnorm


# --------------------------------------------------------------------------
# c-MD  shadow-energy closed form, Eq. 22 (reading G4)
# --------------------------------------------------------------------------
def shadow_charges(chi, u, v, qtot):
    """q[n], lambda from the quasi-diagonal system Eq. 22 given v = ke*phi[n]:
         u_i q_i + lambda = -chi_i - v_i ,  sum q = Qtot."""
    chi = _f64(chi); u = _f64(u); v = _f64(v)
    lam = -(float(qtot) + np.sum((chi + v) / u)) / np.sum(1.0 / u)
    q = -(chi + v + lam) / u
    return q, float(lam)


# --------------------------------------------------------------------------
# c-MD  shadow XL-BOMD step (Eqs. 19-27; readings DESIGN.md R-MD)
#       Integrator constants are not in the paper: PARITY UNPINNED for those.
#       Pinned: Eq. 22 rows, sum q = Qtot, forces = -grad of the shadow potential
#       (finite differences), residual 0 and BO forces when n = q_min.
# --------------------------------------------------------------------------
ACC_CONV = 0.00964853321  # (eV/Angstrom)/amu -> Angstrom/fs^2


def harmonic_water(pos, k_oh, r_oh, k_hh, r_hh):
    """Stand-in for V_short (Eq. 14): atoms 3m,3m+1,3m+2 = O,H,H with
    1/2 k_oh (|r_OH|-r_oh)^2 on both O-H bonds and 1/2 k_hh (|r_HH|-r_hh)^2.  Returns V, F."""
    pos = _f64(pos, (-1, 3))
    F = np.zeros_like(pos)
    V = 0.0
    mol = pos.reshape(-1, 3, 3)
    Fm = F.reshape(-1, 3, 3)
    for a, b, k, r0 in ((0, 1, k_oh, r_oh), (0, 2, k_oh, r_oh), (1, 2, k_hh, r_hh)):
        d = mol[:, b] - mol[:, a]
        r = np.linalg.norm(d, axis=1)
        V += 0.5 * k * float(np.sum((r - r0) ** 2))
        f = (k * (r - r0) / r)[:, None] * d       # force on a (towards b when stretched)
        Fm[:, a] += f
        Fm[:, b] -= f
    return V, F


def oo_repulsion(pos, box, k_rep, r0):
    """Second part of the V_short stand-in: a soft-sphere repulsion between the oxygens
    (atoms 3m) of different molecules, V = 1/2 k_rep (r0 - r)^2 for minimum-image r < r0 < L/2, else 0 --
    the role the O-O Lennard-Jones term plays in three-site water models: it keeps unshielded point charges
    from collapsing into each other.  Brute force over all O-O pairs.  Returns V, F (on all atoms)."""
    pos = _f64(pos, (-1, 3)); box = _box(box)
    F = np.zeros_like(pos)
    xo = pos[0::3]
    V = 0.0
    no = xo.shape[0]
    for a in range(no - 1):
        d = xo[a + 1:] - xo[a]
        d -= np.rint(d / box) * box
        r = np.sqrt((d * d).sum(axis=1))
        m = r < r0
        if not m.any():
            continue
        rr = r[m]
        V += 0.5 * k_rep * float(((r0 - rr) ** 2).sum())
        f = (k_rep * (r0 - rr) / rr)[:, None] * d[m]          # pushes b away from a
        idx = np.nonzero(m)[0] + a + 1
        np.add.at(F, 3 * idx, f)
        F[3 * a] -= f.sum(axis=0)
    return V, F


def standin_eval(pos, box, standin):
    """V_short stand-in: harmonic intramolecular terms (standin[0:4]) and, if given, the O-O repulsion
    (standin[4:6] = k_rep, r0)."""
    V, F = harmonic_water(pos, *standin[:4])
    if len(standin) >= 6 and standin[4] != 0.0:
        Vr, Fr = oo_repulsion(pos, box, standin[4], standin[5])
        V += Vr
        F = F + Fr
    return V, F


def shadow_eval(pos, n, chi, u, ke, qtot, box, rc, alpha, grid, order, standin=None):
    """Shadow potential, charges and forces at fixed n (Eqs. 20-22).

    v = ke*phi[n] (one Coulomb potential); q[n], lambda from Eq. 22;
    U = sum q chi + 1/2 sum q^2 u + sum_i (q_i - n_i/2) v_i  (+ stand-in V_short), which is
    Eq. 20 with sum_{j!=i} phi_ij n_j read as the periodic Ewald potential of n;
    F = -grad_R U at fixed q, n = F_Coul[q] - F_Coul[q-n]  (polarisation identity:
    1/2 (2q-n)' Phi n = 1/2 q' Phi q - 1/2 (q-n)' Phi (q-n)), times ke, plus stand-in forces.
    """
    n = _f64(n); chi = _f64(chi); u = _f64(u)
    phi_n = coulomb_pme(pos, n, box, rc, alpha, grid, order)[0]
    v = ke * phi_n
    q, lam = shadow_charges(chi, u, v, qtot)
    U = float(np.dot(q, chi) + 0.5 * np.dot(q * q, u) + np.dot(q - 0.5 * n, v))
    Fq = coulomb_pme(pos, q, box, rc, alpha, grid, order)[1]
    Fd = coulomb_pme(pos, q - n, box, rc, alpha, grid, order)[1]
    F = ke * (Fq - Fd)
    if standin is not None:
        Vs, Fs = standin_eval(pos, box, standin)
        U += Vs
        F = F + Fs
    return dict(U=U, q=q, lam=lam, v=v, F=F, res=q - n)


def kernel_jacobian_apply(pos, w, u, ke, box, rc, alpha, grid, order):
    """J w with J = d(q[n]-n)/dn (Eq. 24).  From Eq. 22,
    q[n] = -(chi + ke Phi n + lambda)/u with lambda fixing sum q, so
    J w = -w - (ke Phi w + dlam)/u,  dlam = -sum_i (ke Phi w)_i/u_i / sum_i 1/u_i."""
    w = _f64(w); u = _f64(u)
    pw = ke * coulomb_pme(pos, w, box, rc, alpha, grid, order)[0]
    dlam = -float(np.sum(pw / u)) / float(np.sum(1.0 / u))
    return -w - (pw + dlam) / u


def gmres_fixed(apply, b, m):
    """m steps of GMRES from a zero initial guess: Arnoldi with modified Gram-Schmidt, then
    the (m+1) x m least-squares problem by numpy.linalg.lstsq.  Returns x_m."""
    b = _f64(b)
    beta = float(np.linalg.norm(b))
    if beta == 0.0:
        return np.zeros_like(b)
    V = [b / beta]
    H = np.zeros((m + 1, m))
    k = m
    for j in range(m):
        w = apply(V[j])
        for i in range(j + 1):
            H[i, j] = float(np.dot(V[i], w))
            w = w - H[i, j] * V[i]
        H[j + 1, j] = float(np.linalg.norm(w))
        if H[j + 1, j] == 0.0:
            k = j + 1
            break
        V.append(w / H[j + 1, j])
    e1 = np.zeros(k + 1); e1[0] = beta
    y = np.linalg.lstsq(H[:k + 1, :k], e1, rcond=None)[0]
    return sum(y[i] * V[i] for i in range(k))


def gmres_tol(apply, b, tol, max_iter, x0=None, diag=None):
    """GMRES (unrestarted, modified Gram-Schmidt) to a relative residual ||b - A x||/||b|| <= tol
    (the paper's convergence measure), at most max_iter Krylov vectors.
    x0: initial guess (its residual costs one more operator application).
    diag: right Jacobi preconditioner ("Jacobi preconditioner is used for regular MD runs as the
    diagonal entries of the matrix are not equal to one"): solves A D^-1 y = b, x = D^-1 y.
    Returns x, operator applications, relative residual (of the least-squares problem)."""
    b = _f64(b)
    bnorm = float(np.linalg.norm(b))
    n_apply = 0
    x_start = np.zeros_like(b) if x0 is None else _f64(x0).copy()
    r0 = b.copy()
    if x0 is not None:
        r0 = b - apply(x_start)
        n_apply += 1
    beta = float(np.linalg.norm(r0))
    if bnorm == 0.0 or beta / bnorm <= tol:
        return x_start, n_apply, (beta / bnorm if bnorm > 0 else 0.0)
    dinv = None if diag is None else 1.0 / _f64(diag)
    V = [r0 / beta]
    H = np.zeros((max_iter + 1, max_iter))
    relres = beta / bnorm
    k = 0
    y = np.zeros(0)
    for j in range(max_iter):
        w = apply(V[j] if dinv is None else dinv * V[j])
        n_apply += 1
        for i in range(j + 1):
            H[i, j] = float(np.dot(V[i], w))
            w = w - H[i, j] * V[i]
        H[j + 1, j] = float(np.linalg.norm(w))
        k = j + 1
        e1 = np.zeros(k + 1); e1[0] = beta
        y, res, *_ = np.linalg.lstsq(H[:k + 1, :k], e1, rcond=None)
        relres = float(np.linalg.norm(H[:k + 1, :k] @ y - e1)) / bnorm
        if relres <= tol or H[j + 1, j] == 0.0:
            break
        V.append(w / H[j + 1, j])
    dx = sum(y[i] * V[i] for i in range(k))
    if dinv is not None:
        dx = dinv * dx
    return x_start + dx, n_apply, relres


def ewald_self_diagonal(box, alpha, tol=1e-17):
    """A_ii of the Ewald matrix (phi[e_i]_i with the uniform background omitted, G11) for r_c < L/2, where
    no image of the atom itself is inside the real-space cutoff: the reciprocal-space self term
    (1/(pi V)) sum_{m != 0} exp(-pi^2 |m/L|^2/alpha^2)/|m/L|^2 minus 2 alpha/sqrt(pi) (Eqs. 4-5)."""
    box = _box(box)
    V = float(np.prod(box))
    mmax = [int(math.ceil(math.sqrt(-math.log(tol)) * alpha * L / math.pi)) for L in box]
    m = np.stack(np.meshgrid(*[np.arange(-k, k + 1) for k in mmax], indexing="ij"), -1).reshape(-1, 3)
    m = m[(m != 0).any(axis=1)]
    mt2 = ((m / box) ** 2).sum(axis=1)
    return float(np.sum(np.exp(-math.pi ** 2 * mt2 / alpha ** 2) / mt2) / (math.pi * V)) - 2.0 * alpha / math.sqrt(math.pi)


def bo_eval(pos, chi, u, ke, qtot, box, rc, alpha, grid, order, standin, tol, max_iter, q_guess=None,
            lam_guess=0.0, jacobi=True):
    """Regular Born-Oppenheimer evaluation (Eqs. 13-19): q_min from Eq. 18 by GMRES to `tol`
    (right Jacobi preconditioner diag(u_i + ke A_ii) on the charge rows, 1 on the constraint row; initial guess
    [q_guess; lam_guess], whose residual costs one operator application), then the forces at FIXED q = q_min,
    F = ke F_Coul[q] + stand-in (Eq. 19: the gradient of U_BO; dq/dR drops out only for converged q -- the
    reason regular MD needs tight tolerances), and U_BO of Eq. 28.
    Coulomb evaluations: GMRES operator applications + 1 (the force evaluation)."""
    chi = _f64(chi); u = _f64(u)
    n = chi.size

    def apply(x):
        phi = coulomb_pme(pos, x[:n], box, rc, alpha, grid, order)[0]
        return np.concatenate([u * x[:n] + ke * phi + x[n], [x[:n].sum()]])

    b = np.concatenate([-chi, [float(qtot)]])
    diag = None
    if jacobi:
        diag = np.concatenate([u + ke * ewald_self_diagonal(box, alpha), [1.0]])
    x0 = None
    if q_guess is not None:
        x0 = np.concatenate([_f64(q_guess), [float(lam_guess)]])
    x, n_apply, relres = gmres_tol(apply, b, tol, max_iter, x0=x0, diag=diag)
    q = x[:n]
    phi, Fc, Ec, _ = coulomb_pme(pos, q, box, rc, alpha, grid, order)
    U = float(np.dot(q, chi) + 0.5 * np.dot(q * q, u) + ke * Ec)
    F = ke * Fc
    if standin is not None:
        Vs, Fs = standin_eval(pos, box, standin)
        U += Vs
        F = F + Fs
    return dict(q=q, lam=float(x[n]), F=F, U=U, evals=n_apply + 1, relres=relres)


def bo_md_step(state, vel, mass, dt, chi, u, ke, qtot, box, rc, alpha, grid, order, standin, tol, max_iter,
               jacobi=True, warm_start=True):
    """One velocity-Verlet step of regular BOMD ("leapfrog velocity Verlet"); the charges of the
    previous step are the solver's initial guess when warm_start."""
    mass = _f64(mass); vel = _f64(vel, (-1, 3))
    vel = vel + 0.5 * dt * ACC_CONV * state["F"] / mass[:, None]
    pos = state["pos"] + dt * vel
    ev = bo_eval(pos, chi, u, ke, qtot, box, rc, alpha, grid, order, standin, tol, max_iter,
                 q_guess=state["q"] if warm_start else None, lam_guess=state.get("lam", 0.0), jacobi=jacobi)
    vel = vel + 0.5 * dt * ACC_CONV * ev["F"] / mass[:, None]
    ekin = 0.5 * float(np.sum(mass[:, None] * vel * vel)) / ACC_CONV
    ev["pos"] = pos
    return ev, vel, ekin


def shadow_md_force_and_ndd(pos, n, chi, u, ke, qtot, box, rc, alpha, grid, order, standin,
                            kappa, krylov_rank, krylov_tol=0.0):
    """Everything the integrator needs at one time level: shadow forces (Eq. 25) and
    dt^2 * ndd from Eq. 27, J (dt^2 ndd) = -kappa (q[n]-n), kappa = dt^2 omega^2, solved by
    `krylov_rank` GMRES steps from zero (the paper's low-rank Krylov approximation of K = J^-1,
    PAPER.md:244-246).  Coulomb evaluations: 1 (v) + 2 (forces) + krylov_rank."""
    ev = shadow_eval(pos, n, chi, u, ke, qtot, box, rc, alpha, grid, order, standin)
    apply = lambda w: kernel_jacobian_apply(pos, w, u, ke, box, rc, alpha, grid, order)
    if krylov_tol > 0.0:      # Table 1's "Sol. Tol.": stop at the relative residual, rank <= krylov_rank
        ev["ndd_dt2"], it, _ = gmres_tol(apply, -kappa * ev["res"], krylov_tol, krylov_rank)
    else:
        ev["ndd_dt2"] = gmres_fixed(apply, -kappa * ev["res"], krylov_rank)
        it = krylov_rank
    # Coulomb evaluations of the METHOD at this time level (reading G16): potential + field of n, field of q - n,
    # one per Krylov vector (this oracle itself spends one more, computing F_Coul[q] and F_Coul[q-n] separately)
    ev["evals"] = 2 + it
    return ev


def xl_n_update(nh, ndd_dt2, alpha_diss, c):
    """Verlet step with dissipation for the extended charges (DESIGN.md R-MD; the form of the
    integration the paper cites for Eq. 27):
        n(t+dt) = 2 n(t) - n(t-dt) + dt^2 ndd(t) + alpha_diss * sum_{k=0}^{5} c_k n(t - k dt),
    nh[k] = n(t - k dt), k = 0..5.  alpha_diss = 0 is the plain time-reversible Verlet step."""
    nh = np.asarray(nh, dtype=np.float64)
    diss = np.zeros_like(nh[0])
    for k in range(6):
        diss = diss + float(c[k]) * nh[k]
    return 2.0 * nh[0] - nh[1] + _f64(ndd_dt2) + float(alpha_diss) * diss


def shadow_md_init(pos, n0, chi, u, ke, qtot, box, rc, alpha, grid, order, standin, kappa,
                   krylov_rank, krylov_tol=0.0):
    """History rows 0..5 = n0 (PAPER.md is silent on the start: DESIGN.md R-MD), row 6 = dt^2 ndd."""
    n0 = _f64(n0)
    ev = shadow_md_force_and_ndd(pos, n0, chi, u, ke, qtot, box, rc, alpha, grid, order, standin,
                                 kappa, krylov_rank, krylov_tol)
    nhist = np.vstack([np.tile(n0, (6, 1)), ev["ndd_dt2"][None, :]])
    return dict(pos=_f64(pos, (-1, 3)).copy(), nhist=nhist, F=ev["F"], U=ev["U"], q=ev["q"],
                res=ev["res"])


def shadow_md_step(state, vel, mass, dt, chi, u, ke, qtot, box, rc, alpha, grid, order, standin,
                   kappa, alpha_diss, c, krylov_rank, krylov_tol=0.0):
    """One velocity-Verlet step for R and one Verlet step with dissipation for n
    (R-MD):  n(t+dt) = 2 n(t) - n(t-dt) + dt^2 ndd(t) + alpha_diss * sum_k c_k n(t - k dt).
    Returns the new state, new velocities and the kinetic energy (eV)."""
    pos = state["pos"]; nh = state["nhist"]
    mass = _f64(mass); vel = _f64(vel, (-1, 3))
    a = ACC_CONV * state["F"] / mass[:, None]
    vel = vel + 0.5 * dt * a
    pos = pos + dt * vel
    n_new = xl_n_update(nh[0:6], nh[6], alpha_diss, c)
    ev = shadow_md_force_and_ndd(pos, n_new, chi, u, ke, qtot, box, rc, alpha, grid, order,
                                 standin, kappa, krylov_rank, krylov_tol)
    nhist = np.vstack([n_new[None, :], nh[0:5], ev["ndd_dt2"][None, :]])
    a = ACC_CONV * ev["F"] / mass[:, None]
    vel = vel + 0.5 * dt * a
    ekin = 0.5 * float(np.sum(mass[:, None] * vel * vel)) / ACC_CONV
    new = dict(pos=pos, nhist=nhist, F=ev["F"], U=ev["U"], q=ev["q"], res=ev["res"], evals=ev["evals"])
    return new, vel, ekin
