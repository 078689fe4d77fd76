"""Pins of the oracle's shadow XL-BOMD ingredients (CPU only).

The n(t) integrator's constants are not in the paper (parity unpinned, DESIGN.md R-MD); what the
paper and the mathematics do fix is pinned here: forces are minus the gradient of the shadow
potential of Eq. 21 (finite differences with q re-relaxed at every displaced geometry), Eq. 24's
Jacobian is the derivative of q[n]-n, the shadow potential touches the regular BO potential at
n = q_min (residual 0, equal forces), GMRES is checked against scipy, and a short NVE run
conserves the shadow total energy.
"""
import numpy as np
import pytest
from scipy.sparse.linalg import LinearOperator, gmres

import oracle
from paper_2503_21176_b200 import workloads as W

KE = oracle.KE_EV_A
STANDIN = (48.0, 0.9572, 10.0, 1.5139)


def small_water(nlat=3, seed=7):
    L = 3.1066 * nlat
    pos, q = W.water_box(nlat, L, seed)
    n = len(q)
    chi, u = W.qeq_params_water_pd(n)
    geo = dict(box=[L] * 3, rc=0.48 * L, alpha=0.75, grid=16, order=6)
    return pos, q, chi.astype(float), u.astype(float), geo


def test_standin_forces_are_minus_gradient():
    pos, *_ = small_water(2)
    V, F = oracle.harmonic_water(pos, *STANDIN)
    for i, k in ((0, 0), (4, 2), (8, 1)):
        h = 1e-6
        p = pos.copy(); p[i, k] += h; Vp = oracle.harmonic_water(p, *STANDIN)[0]
        p[i, k] -= 2 * h; Vm = oracle.harmonic_water(p, *STANDIN)[0]
        assert abs(-(Vp - Vm) / (2 * h) - F[i, k]) < 1e-6 * max(1.0, abs(F[i, k]))
    assert np.abs(F.reshape(-1, 3, 3).sum(axis=1)).max() < 1e-12     # no net force per molecule


def test_shadow_forces_are_minus_gradient_of_shadow_potential():
    pos, q0, chi, u, geo = small_water(2)
    rng = np.random.default_rng(1)
    n = q0 + 0.05 * rng.normal(size=len(q0))
    ev = oracle.shadow_eval(pos, n, chi, u, KE, 0.0, standin=STANDIN, **geo)
    assert abs(ev["q"].sum()) < 1e-12
    assert np.abs(u * ev["q"] + ev["lam"] + chi + ev["v"]).max() < 1e-10      # Eq. 22 rows
    for i, k in ((0, 0), (7, 1), (13, 2)):
        h = 1e-5
        p = pos.copy(); p[i, k] += h
        Up = oracle.shadow_eval(p, n, chi, u, KE, 0.0, standin=STANDIN, **geo)["U"]
        p[i, k] -= 2 * h
        Um = oracle.shadow_eval(p, n, chi, u, KE, 0.0, standin=STANDIN, **geo)["U"]
        fd = -(Up - Um) / (2 * h)
        assert abs(fd - ev["F"][i, k]) < 2e-6 * max(1.0, abs(fd)), (fd, ev["F"][i, k])


def test_jacobian_is_derivative_of_residual_and_gmres_matches_scipy():
    pos, q0, chi, u, geo = small_water(2)
    rng = np.random.default_rng(2)
    N = len(q0)
    n = q0 + 0.05 * rng.normal(size=N)
    w = rng.normal(size=N)
    res = lambda nn: oracle.shadow_eval(pos, nn, chi, u, KE, 0.0, **geo)["res"]
    Jw = oracle.kernel_jacobian_apply(pos, w, u, KE, **geo)
    assert np.abs((res(n + 0.5 * w) - res(n - 0.5 * w)) - Jw).max() < 1e-9   # q[n] is affine in n
    assert abs(Jw.sum() + w.sum()) < 1e-10          # d(sum q)/dn = 0  =>  1'Jw = -1'w
    apply = lambda v: oracle.kernel_jacobian_apply(pos, v, u, KE, **geo)
    b = -1.82 * res(n)
    for m in (2, 4):
        x = oracle.gmres_fixed(apply, b, m)
        xs, _ = gmres(LinearOperator((N, N), matvec=apply), b, x0=np.zeros(N), restart=m, maxiter=1,
                      rtol=1e-30, atol=0.0)
        assert np.abs(x - xs).max() < 1e-9 * np.abs(xs).max()
    xf = oracle.gmres_fixed(apply, b, N)
    assert np.abs(apply(xf) - b).max() < 1e-8 * np.abs(b).max()


def test_shadow_touches_regular_bo_at_qmin():
    pos, q0, chi, u, geo = small_water(2)
    A = oracle.coulomb_matrix_pme(pos, **geo)
    qmin, lam = oracle.qeq_dense_solve(A, chi, u, KE, 0.0)
    ev = oracle.shadow_eval(pos, qmin, chi, u, KE, 0.0, **geo)
    assert np.abs(ev["res"]).max() < 1e-10                     # q[q_min] = q_min
    assert abs(ev["lam"] - lam) < 1e-9
    F_bo = KE * oracle.coulomb_pme(pos, qmin, **geo)[1]
    assert np.abs(ev["F"] - F_bo).max() < 1e-9
    E_bo = qmin @ chi + 0.5 * qmin @ (u * qmin) + 0.5 * KE * qmin @ A @ qmin   # Eq. 13
    assert abs(ev["U"] - E_bo) < 1e-9


def aligned_water(nlat=2, seed=3):
    """Waters on a lattice, all with the same orientation (+ small jitter): no close intermolecular
    contacts, so the point-charge model without V_short's repulsion stays bound for a short run."""
    rng = np.random.default_rng(seed)
    L = 3.1066 * nlat
    frame = W._water_frame()
    o = (np.stack(np.meshgrid(*[np.arange(nlat)] * 3, indexing="ij"), -1).reshape(-1, 3) + 0.5) * (L / nlat)
    pos = (o[:, None, :] + frame[None, :, :]).reshape(-1, 3) + rng.normal(0, 0.02, (3 * nlat ** 3, 3))
    n = len(pos)
    chi, u = W.qeq_params_water_pd(n)
    geo = dict(box=[L] * 3, rc=0.48 * L, alpha=0.75, grid=16, order=6)
    return pos, chi.astype(float), u.astype(float), geo


def test_short_nve_run_conserves_shadow_energy():
    pos, chi, u, geo = aligned_water(2)
    q0 = np.zeros(len(pos))
    A = oracle.coulomb_matrix_pme(pos, **geo)
    qmin, _ = oracle.qeq_dense_solve(A, chi, u, KE, 0.0)
    n_atoms = len(q0)
    mass = W.masses_water(n_atoms).astype(float)
    vel = W.velocities(mass).astype(float)
    c = [-6.0, 14.0, -8.0, -3.0, 4.0, -1.0]
    kw = dict(chi=chi, u=u, ke=KE, qtot=0.0, standin=STANDIN, kappa=1.82, krylov_rank=4, **geo)
    st = oracle.shadow_md_init(pos, qmin, **kw)
    e, k = [], []
    for _ in range(30):
        st, vel, ekin = oracle.shadow_md_step(st, vel, mass, 0.5, alpha_diss=0.018, c=c, **kw)
        e.append(st["U"] + ekin)
        k.append(ekin)
        assert abs(st["q"].sum()) < 1e-10
        assert np.abs(st["res"]).max() < 0.01
    e, k = np.array(e), np.array(k)
    # kinetic and potential energy exchange O(0.1-1 eV) while their sum stays flat
    assert np.ptp(k) > 0.3
    assert e.std() < 0.02 * np.ptp(k), (e.std(), np.ptp(k))


# ---- the n(t) integrator (oracle.xl_n_update): what the mathematics fixes ---------------------------
# kappa, alpha_diss and c_k are not printed in the paper (DESIGN.md R-MD); they are the K = 5 set of the
# XL-BOMD literature it cites.  What can be checked without that literature: the dissipation term must
# not move a stationary n (sum c = 0), must be invisible to time reversal up to high order in dt (the odd
# moments sum k^p c_k, p = 1, 3, 5 vanish -- the design condition that determines such a set up to its
# scale and one free parameter), the step at alpha_diss = 0 is exactly reversible, and the homogeneous
# recursion with the exact kernel (dt^2 ndd = -kappa (n - q)) must be stable: all roots of its
# characteristic polynomial inside the closed unit disc, strictly inside when alpha_diss > 0.
XL_KAPPA, XL_ALPHA, XL_C = 1.82, 0.018, [-6.0, 14.0, -8.0, -3.0, 4.0, -1.0]


def test_xl_coefficients_moments():
    c = np.array(XL_C)
    k = np.arange(6.0)
    assert c.sum() == 0.0
    for p in (1, 3, 5):
        assert (k ** p * c).sum() == 0.0, p
    assert (k ** 2 * c).sum() != 0.0          # the even moment carries the dissipation
    # stationary n, no acceleration: stays put for any alpha_diss
    n = np.array([0.3, -0.7, 0.4])
    assert np.abs(oracle.xl_n_update(np.tile(n, (6, 1)), np.zeros(3), 0.5, XL_C) - n).max() < 1e-15


def test_xl_step_is_time_reversible_without_dissipation():
    rng = np.random.default_rng(0)
    nh = rng.normal(size=(6, 50))
    acc = rng.normal(size=50) * 0.1
    fwd = oracle.xl_n_update(nh, acc, 0.0, XL_C)                       # n(t+dt)
    back_hist = np.vstack([nh[0:1], fwd[None, :], nh[1:5]])            # time reversed: n(t), n(t+dt), ...
    back = oracle.xl_n_update(back_hist, acc, 0.0, XL_C)               # same acceleration at t
    assert np.abs(back - nh[1]).max() < 1e-15
    # with dissipation the reversed step does NOT return (the term breaks time reversal on purpose)
    fwd_d = oracle.xl_n_update(nh, acc, XL_ALPHA, XL_C)
    back_d = oracle.xl_n_update(np.vstack([nh[0:1], fwd_d[None, :], nh[1:5]]), acc, XL_ALPHA, XL_C)
    assert np.abs(back_d - nh[1]).max() > 1e-4


def _char_roots(kappa, alpha, c):
    # n_{j+1} = (2 - kappa) n_j - n_{j-1} + alpha sum_k c_k n_{j-k}   =>   polynomial in z of degree 6
    p = [1.0, -(2.0 - kappa + alpha * c[0]), 1.0 - alpha * c[1], -alpha * c[2], -alpha * c[3], -alpha * c[4],
         -alpha * c[5]]
    return np.roots(p)


def test_xl_recursion_is_stable_and_damped():
    r0 = _char_roots(XL_KAPPA, 0.0, XL_C)
    assert np.abs(np.abs(r0[np.abs(r0) > 1e-8]) - 1.0).max() < 1e-12      # undamped Verlet: on the unit circle
    r = _char_roots(XL_KAPPA, XL_ALPHA, XL_C)
    rho = np.abs(r).max()
    assert rho < 0.92                                        # strictly inside: noise in n is damped
    # sign or index slips in c, or kappa beyond the Verlet limit, leave the disc
    assert np.abs(_char_roots(XL_KAPPA, XL_ALPHA, [-x for x in XL_C])).max() > 1.0
    assert np.abs(_char_roots(XL_KAPPA, XL_ALPHA, XL_C[::-1])).max() > 1.0
    assert np.abs(_char_roots(4.2, XL_ALPHA, XL_C)).max() > 1.0
    # the oracle's recursion itself, run on the exact-kernel model problem dt^2 ndd = -kappa (n - q):
    # the error decays at the rate of the largest root
    q = np.array([0.4, -0.1])
    nh = np.tile(q + np.array([0.05, -0.02]), (6, 1))
    err = []
    for _ in range(120):
        n_new = oracle.xl_n_update(nh, -XL_KAPPA * (nh[0] - q), XL_ALPHA, XL_C)
        nh = np.vstack([n_new[None, :], nh[0:5]])
        err.append(np.abs(n_new - q).max())
    err = np.array(err)
    assert err[-1] < 1e-4 * err[0]
    rate = (err[100:120].max() / err[40:60].max()) ** (1.0 / 60.0)
    assert abs(rate - rho) < 0.02, (rate, rho)


# ---- regular BOMD ingredients (NEXT-2) ----------------------------------------
def test_oo_repulsion_forces_are_minus_gradient_and_compact():
    pos, *_ , geo = small_water(3)
    box = geo["box"]
    V, F = oracle.oo_repulsion(pos, box, 10.0, 3.3)
    assert V > 0.0
    assert np.abs(F[1::3]).max() == 0.0 and np.abs(F[2::3]).max() == 0.0        # oxygens only
    assert np.abs(F.sum(axis=0)).max() < 1e-12
    for i, k in ((0, 0), (3, 1), (12, 2)):
        h = 1e-6
        p = pos.copy(); p[i, k] += h; Vp = oracle.oo_repulsion(p, box, 10.0, 3.3)[0]
        p[i, k] -= 2 * h; Vm = oracle.oo_repulsion(p, box, 10.0, 3.3)[0]
        assert abs(-(Vp - Vm) / (2 * h) - F[i, k]) < 1e-6 * max(1.0, abs(F[i, k]))
    # translation by a box vector of one molecule changes nothing (minimum image); r0 below the closest O-O: zero
    p = pos.copy(); p[3:6] += np.array(box) * np.array([1, -2, 0])
    assert abs(oracle.oo_repulsion(p, box, 10.0, 3.3)[0] - V) < 1e-12
    do = pos[0::3][:, None, :] - pos[0::3][None, :, :]
    do -= np.rint(do / np.array(box)) * np.array(box)
    rmin = np.sqrt((do ** 2).sum(-1))[np.triu_indices(len(pos) // 3, 1)].min()
    assert oracle.oo_repulsion(pos, box, 10.0, 0.99 * rmin)[0] == 0.0


def test_gmres_tol_matches_scipy_with_jacobi_and_initial_guess():
    rng = np.random.default_rng(3)
    N = 40
    B = rng.normal(size=(N, N)); A = B @ B.T / N + np.diag(rng.uniform(1, 30, N))
    b = rng.normal(size=N)
    x0 = rng.normal(size=N) * 0.1
    d = np.diag(A).copy()
    ap = lambda v: A @ v
    for tol in (1e-2, 1e-6):
        x, it, rel = oracle.gmres_tol(ap, b, tol, N, x0=x0, diag=d)
        assert np.linalg.norm(b - A @ x) / np.linalg.norm(b) <= tol * 1.0001
        assert abs(rel - np.linalg.norm(b - A @ x) / np.linalg.norm(b)) < 1e-10
        # scipy's GMRES on the right-preconditioned operator with the same start builds the same Krylov space:
        # after the same number of vectors the iterates agree
        nk = it - 1                                                 # one application went into the guess's residual
        Ar = LinearOperator((N, N), matvec=lambda y: A @ (y / d))
        ys, _ = gmres(Ar, b - A @ x0, x0=np.zeros(N), restart=nk, maxiter=1, rtol=1e-30, atol=0.0)
        assert np.abs(x - (x0 + ys / d)).max() < 1e-9
    # the preconditioner pays: fewer vectors than without it on this badly scaled matrix
    assert oracle.gmres_tol(ap, b, 1e-6, N, diag=d)[1] < oracle.gmres_tol(ap, b, 1e-6, N)[1]


def test_ewald_self_diagonal_is_the_diagonal_of_the_coulomb_matrix():
    # cubic box: xi/L + pi/(V alpha^2) with xi = -2.8372974795 (the pin of test_oracle_pins), any alpha with
    # erfc(alpha L) negligible; and equal to the diagonal of the direct-Ewald matrix for a non-cubic box
    L, a = 9.0, 0.9
    assert abs(oracle.ewald_self_diagonal([L] * 3, a) - (-2.8372974795 / L + np.pi / (L ** 3 * a * a))) < 1e-9
    box = [8.0, 9.5, 11.0]
    phi, _, _ = oracle.ewald_direct(np.array([[1.0, 2.0, 3.0]]), np.array([1.0]), box, 1.1)
    assert abs(oracle.ewald_self_diagonal(box, 1.1) - phi[0]) < 1e-9


def test_bo_forces_are_minus_gradient_of_u_bo_and_match_shadow_at_qmin():
    pos, q0, chi, u, geo = small_water(2)
    st6 = STANDIN + (10.0, 3.3)
    ev = oracle.bo_eval(pos, chi, u, KE, 0.0, standin=st6, tol=1e-13, max_iter=30, **geo)
    assert ev["relres"] <= 1e-13 and abs(ev["q"].sum()) < 1e-12
    A = oracle.coulomb_matrix_pme(pos, **geo)
    qd, lamd = oracle.qeq_dense_solve(A, chi, u, KE, 0.0)
    assert np.abs(ev["q"] - qd).max() < 1e-10 and abs(ev["lam"] - lamd) < 1e-9
    for i, k in ((0, 0), (7, 1), (13, 2)):
        h = 1e-5
        p = pos.copy(); p[i, k] += h
        Up = oracle.bo_eval(p, chi, u, KE, 0.0, standin=st6, tol=1e-13, max_iter=30, **geo)["U"]
        p[i, k] -= 2 * h
        Um = oracle.bo_eval(p, chi, u, KE, 0.0, standin=st6, tol=1e-13, max_iter=30, **geo)["U"]
        fd = -(Up - Um) / (2 * h)
        assert abs(fd - ev["F"][i, k]) < 2e-6 * max(1.0, abs(fd)), (fd, ev["F"][i, k])
    sh = oracle.shadow_eval(pos, ev["q"], chi, u, KE, 0.0, standin=st6, **geo)
    assert np.abs(sh["F"] - ev["F"]).max() < 1e-8 and abs(sh["U"] - ev["U"]) < 1e-8
    # a warm start from the solution needs one application (its residual) and no Krylov vector
    ev2 = oracle.bo_eval(pos, chi, u, KE, 0.0, standin=st6, tol=1e-8, max_iter=30, q_guess=ev["q"],
                         lam_guess=ev["lam"], **geo)
    assert ev2["evals"] == 2


def test_bo_md_conserves_energy_when_converged_and_drifts_when_loose():
    """The paper's Table 1 in miniature: regular BOMD conserves energy with a tight solver and
    not with a loose one, at more Coulomb evaluations per step than shadow MD needs."""
    pos, chi, u, geo = aligned_water(2)
    st6 = STANDIN + (10.0, 2.9)
    mass = W.masses_water(len(pos)).astype(float)
    out = {}
    for tol in (1e-8, 1e-2):
        ev = oracle.bo_eval(pos, chi, u, KE, 0.0, standin=st6, tol=1e-10, max_iter=40, **geo)
        st = dict(pos=pos.copy(), F=ev["F"], q=ev["q"], lam=ev["lam"])
        vel = W.velocities(mass).astype(float)
        e, evals, k = [], [], []
        for _ in range(25):
            st, vel, ekin = oracle.bo_md_step(st, vel, mass, 0.5, chi, u, KE, 0.0, standin=st6, tol=tol, max_iter=40, **geo)
            e.append(st["U"] + ekin); evals.append(st["evals"]); k.append(ekin)
        out[tol] = (np.std(e), np.mean(evals), np.ptp(k))
    # converged charges: the total energy holds to the Verlet error of the stiff bonds (1 % of the kinetic/potential
    # exchange at 0.5 fs); tol 1e-2: the warm-started solver updates the charges only now and then, the forces are
    # not the gradient of any potential and the energy wanders by tens of times more -- at a quarter of the cost
    assert out[1e-8][0] < 0.02 * out[1e-8][2] and out[1e-8][1] > 3 * out[1e-2][1]
    assert out[1e-2][0] > 10 * out[1e-8][0]
