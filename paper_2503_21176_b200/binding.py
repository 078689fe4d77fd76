"""Thin ctypes binding of libsqeq (include/sqeq.h): argument marshalling only.

Every step of the path runs in the CUDA library; PyTorch supplies device memory and streams.
There is no fallback: `load()` raises if the library is missing, and every call raises
`SqeqError` with the library's message on a non-zero return code.
"""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsqeq.so")

OK, EINVAL, ECAPACITY, ECUDA, ECUFFT, ENOTCONV, ENOMEM = 0, -1, -2, -3, -4, -5, -6
STAGES = ["nl_bin", "nl_pairs", "prep", "real", "spread", "fft_fwd", "influence", "fft_inv",
          "gather", "assemble", "krylov"]

_lib = None


class SqeqError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libsqeq error {code}: {msg}")
        self.code = code


class MdParams(ctypes.Structure):
    _fields_ = [("dt", ctypes.c_double), ("ke", ctypes.c_double), ("total_charge", ctypes.c_double),
                ("rc", ctypes.c_double), ("alpha", ctypes.c_double), ("grid", ctypes.c_int * 3),
                ("order", ctypes.c_int), ("krylov_rank", ctypes.c_int),
                ("k_oh", ctypes.c_double), ("r_oh", ctypes.c_double),
                ("k_hh", ctypes.c_double), ("r_hh", ctypes.c_double),
                ("kappa", ctypes.c_double), ("alpha_diss", ctypes.c_double),
                ("c", ctypes.c_double * 7),
                ("krylov_tol", ctypes.c_double), ("k_rep", ctypes.c_double), ("r_rep", ctypes.c_double)]


def load():
    """Load libsqeq.so (built in-tree by `python -m paper_2503_21176_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2503_21176_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, i64, dbl, cint = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
    dp = ctypes.POINTER(ctypes.c_double)
    ip = ctypes.POINTER(ctypes.c_int)
    L.sqeq_version.restype = ctypes.c_char_p
    L.sqeq_last_error.restype = ctypes.c_char_p
    L.sqeq_last_error.argtypes = [vp]
    L.sqeq_create.argtypes = [ctypes.POINTER(vp), cint, vp]
    L.sqeq_destroy.argtypes = [vp]
    L.sqeq_nl_build.argtypes = [vp, i64, vp, dp, dbl, ctypes.POINTER(vp)]
    L.sqeq_nl_count.argtypes = [vp, ctypes.POINTER(i64)]
    L.sqeq_nl_export.argtypes = [vp, vp, vp, vp, vp]
    L.sqeq_nl_export_ellpack.argtypes = [vp, vp, cint, vp, vp, vp]
    L.sqeq_nl_export_coo.argtypes = [vp, vp, vp, vp, vp]
    L.sqeq_nl_info.argtypes = [vp, ip, ctypes.POINTER(i64), ip]
    L.sqeq_nl_entry_bytes.argtypes = [vp, ip]
    L.sqeq_nl_layout.argtypes = [vp, ctypes.POINTER(i64), ip, ip]
    L.sqeq_nl_max_drift.argtypes = [vp, vp, i64, vp, dp]
    L.sqeq_nl_max_drift_ahead.argtypes = [vp, vp, i64, vp, vp, dbl, dp]
    L.sqeq_nl_free.argtypes = [vp]
    L.sqeq_coulomb.argtypes = [vp, vp, i64, vp, vp, dp, dbl, dbl, ip, cint, vp, vp, dp]
    L.sqeq_coulomb_host_submit.argtypes = [vp, cint, vp, i64, vp, vp, dp, dbl, dbl, ip, cint, vp, vp, cint]
    L.sqeq_coulomb_host_wait.argtypes = [vp, cint, dp]
    L.sqeq_coulomb_enqueue.argtypes = [vp, vp, i64, vp, vp, dp, dbl, dbl, ip, cint, vp, vp, cint]
    L.sqeq_energy_fetch.argtypes = [vp, dp]
    L.sqeq_coulomb_ewald.argtypes = [vp, vp, i64, vp, vp, dp, dbl, dbl, ip, vp, vp, dp]
    L.sqeq_ewald_params.argtypes = [dp, dbl, dbl, dp, ip, ip]
    L.sqeq_energy_noalloc.argtypes = [cint, vp, i64, vp, vp, vp]
    L.sqeq_geometry_set.argtypes = [vp, vp, i64, vp, dp, dbl, dbl, ip, cint]
    L.sqeq_coulomb_fixed.argtypes = [vp, i64, vp, vp, vp, cint]
    L.sqeq_coulomb_fixed_batch.argtypes = [vp, i64, cint, vp, vp]
    L.sqeq_coulomb_host.argtypes = [vp, vp, i64, vp, vp, dp, dbl, dbl, ip, cint, vp, vp, dp]
    L.sqeq_coulomb_parts.argtypes = [vp, vp, i64, vp, vp, vp, vp, dp]
    L.sqeq_pme_grid.argtypes = [vp, cint, vp]
    L.sqeq_qeq_solve.argtypes = [vp, vp, i64, vp, dp, dbl, dbl, ip, cint, dbl, vp, vp, dbl, dbl, cint,
                                 cint, vp, dp, ip, dp]
    L.sqeq_qeq_solve_pc.argtypes = [vp, vp, i64, vp, dp, dbl, dbl, ip, cint, dbl, vp, vp, dbl, dbl, cint,
                                    cint, cint, vp, dbl, vp, dp, ip, dp]
    L.sqeq_bomd_init.argtypes = [vp, vp, i64, vp, dp, ctypes.POINTER(MdParams), vp, vp, dbl, cint, cint,
                                 vp, dp, vp, dp]
    L.sqeq_bomd_step.argtypes = [vp, vp, i64, vp, vp, vp, dp, ctypes.POINTER(MdParams), vp, vp, dbl, cint, cint,
                                 cint, vp, dp, vp, dp]
    L.sqeq_shadow_md_init.argtypes = [vp, vp, i64, vp, dp, ctypes.POINTER(MdParams), vp, vp, dbl, cint,
                                      vp, vp, dp]
    L.sqeq_shadow_md_step.argtypes = [vp, vp, i64, vp, vp, vp, dp, ctypes.POINTER(MdParams), vp, vp,
                                      vp, vp, dp]
    L.sqeq_shadow_md_run.argtypes = [vp, ctypes.POINTER(vp), i64, vp, vp, vp, dp, ctypes.POINTER(MdParams), vp, vp,
                                     vp, vp, cint, dbl, dbl, dp]
    L.sqeq_profile_enable.argtypes = [vp, cint]
    L.sqeq_profile_reset.argtypes = [vp]
    L.sqeq_profile_read.argtypes = [vp, cint, dp, ctypes.POINTER(i64)]
    L.sqeq_set_option.argtypes = [vp, ctypes.c_char_p, cint]
    L.sqeq_launch_count.argtypes = [vp, ctypes.POINTER(i64), cint]
    _lib = L
    return L


def _box(box):
    b = np.ascontiguousarray(np.asarray(box, dtype=np.float64).reshape(-1))
    if b.size == 1:
        b = np.repeat(b, 3)
    return (ctypes.c_double * 3)(*b.tolist())


def _grid(grid):
    g = np.asarray(grid, dtype=np.int64).reshape(-1)
    if g.size == 1:
        g = np.repeat(g, 3)
    return (ctypes.c_int * 3)(*[int(v) for v in g])


def _ptr(t, dtype, numel=None):
    if t is None:
        return None
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dtype, \
        f"expected a contiguous CUDA tensor of {dtype}"
    if numel is not None:
        assert t.numel() == numel, f"expected {numel} elements, got {t.numel()}"
    return ctypes.c_void_p(t.data_ptr())


class NeighbourList:
    """Handle of a device neighbour list (sqeq_nlist*)."""

    def __init__(self, ctx, handle, n, box, cutoff):
        self.ctx, self.handle, self.n, self.box, self.cutoff = ctx, handle, n, box, cutoff

    def count(self):
        c = ctypes.c_int64()
        self.ctx._check(load().sqeq_nl_count(self.handle, ctypes.byref(c)))
        return c.value

    def info(self):
        nc = (ctypes.c_int * 3)()
        nd = ctypes.c_int64()
        mr = ctypes.c_int()
        self.ctx._check(load().sqeq_nl_info(self.handle, nc, ctypes.byref(nd), ctypes.byref(mr)))
        eb = ctypes.c_int()
        self.ctx._check(load().sqeq_nl_entry_bytes(self.handle, ctypes.byref(eb)))
        ns = ctypes.c_int64()
        sh, mp = ctypes.c_int(), ctypes.c_int()
        self.ctx._check(load().sqeq_nl_layout(self.handle, ctypes.byref(ns), ctypes.byref(sh), ctypes.byref(mp)))
        return dict(ncell=list(nc), n_directed=nd.value, max_row=mr.value, entry_bytes=eb.value,
                    n_slots=ns.value, entry_shift=sh.value, max_neighbourhood=mp.value)

    def max_drift(self, pos):
        """Largest displacement since the build (rebuild when it reaches skin/2)."""
        d = ctypes.c_double()
        self.ctx._check(load().sqeq_nl_max_drift(self.ctx.handle, self.handle, self.n,
                                                 _ptr(pos, torch.float32, 3 * self.n), ctypes.byref(d)))
        return d.value

    def max_drift_ahead(self, pos, vel, dt):
        """Largest displacement since the build after moving on by vel * dt (rebuild before the step if >= skin/2)."""
        d = ctypes.c_double()
        self.ctx._check(load().sqeq_nl_max_drift_ahead(self.ctx.handle, self.handle, self.n,
                                                       _ptr(pos, torch.float32, 3 * self.n),
                                                       _ptr(vel, torch.float32, 3 * self.n), float(dt), ctypes.byref(d)))
        return d.value

    def export(self):
        """Canonical (i, j, shift) arrays on the device: unique pairs i<j sorted by (i,j)."""
        m = self.count()
        dev = self.ctx.device
        i = torch.empty(m, dtype=torch.int32, device=dev)
        j = torch.empty(m, dtype=torch.int32, device=dev)
        s = torch.empty((m, 3), dtype=torch.int8, device=dev)
        self.ctx._check(load().sqeq_nl_export(self.ctx.handle, self.handle,
                                              ctypes.c_void_p(i.data_ptr()), ctypes.c_void_p(j.data_ptr()),
                                              ctypes.c_void_p(s.data_ptr())))
        return i, j, s

    def export_ellpack(self, K=None):
        """ELLPACK rows [n][K] (padded with -1), shifts [n][K][3], counts [n] on the device."""
        K = self.info()["max_row"] if K is None else K
        K = max(int(K), 1)
        dev = self.ctx.device
        nbr = torch.empty((self.n, K), dtype=torch.int32, device=dev)
        sh = torch.empty((self.n, K, 3), dtype=torch.int8, device=dev)
        cnt = torch.empty(self.n, dtype=torch.int32, device=dev)
        self.ctx._check(load().sqeq_nl_export_ellpack(self.ctx.handle, self.handle, K, ctypes.c_void_p(nbr.data_ptr()),
                                                      ctypes.c_void_p(sh.data_ptr()), ctypes.c_void_p(cnt.data_ptr())))
        return nbr, sh, cnt

    def export_coo(self):
        """Directed COO (every pair both ways) sorted by (i, j) on the device."""
        m = 2 * self.count()
        dev = self.ctx.device
        i = torch.empty(m, dtype=torch.int32, device=dev)
        j = torch.empty(m, dtype=torch.int32, device=dev)
        s = torch.empty((m, 3), dtype=torch.int8, device=dev)
        self.ctx._check(load().sqeq_nl_export_coo(self.ctx.handle, self.handle, ctypes.c_void_p(i.data_ptr()),
                                                  ctypes.c_void_p(j.data_ptr()), ctypes.c_void_p(s.data_ptr())))
        return i, j, s

    def free(self):
        if self.handle:
            load().sqeq_nl_free(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Context:
    """sqeq_ctx*: bound to one device and one stream (default: torch's current stream)."""

    def __init__(self, device=0, stream=None):
        L = load()
        if not torch.cuda.is_available():
            raise SqeqError(ECUDA, "no CUDA device: libsqeq has no CPU fallback")
        self.device = torch.device("cuda", device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        h = ctypes.c_void_p()
        rc = L.sqeq_create(ctypes.byref(h), device, ctypes.c_void_p(stream.cuda_stream))
        if rc != OK:
            raise SqeqError(rc, L.sqeq_last_error(None).decode())
        self.handle = h

    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise SqeqError(rc, load().sqeq_last_error(self.handle).decode())
        return rc

    def close(self):
        if self.handle:
            load().sqeq_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- nl_build(pos, box, cutoff) -> pair list
    def nl_build(self, pos, box, cutoff):
        n = pos.shape[0]
        h = ctypes.c_void_p()
        self._check(load().sqeq_nl_build(self.handle, n, _ptr(pos, torch.float32, 3 * n), _box(box),
                                         float(cutoff), ctypes.byref(h)))
        return NeighbourList(self, h, n, box, cutoff)

    # ---- coulomb(pos, q, box, alpha, grid, order) -> per-atom potential, forces, energy
    def coulomb(self, nl, pos, q, box, rc, alpha, grid, order=6, want_force=True, want_energy=True,
                phi=None, force=None):
        n = pos.shape[0]
        if phi is None:
            phi = torch.empty(n, dtype=torch.float32, device=self.device)
        if want_force and force is None:
            force = torch.empty((n, 3), dtype=torch.float32, device=self.device)
        e = ctypes.c_double()
        self._check(load().sqeq_coulomb(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                        _ptr(q, torch.float32, n), _box(box), float(rc), float(alpha),
                                        _grid(grid), int(order), _ptr(phi, torch.float32, n),
                                        _ptr(force, torch.float32, 3 * n) if want_force else None,
                                        ctypes.byref(e) if want_energy else None))
        return phi, (force if want_force else None), (e.value if want_energy else None)

    def coulomb_ewald(self, nl, pos, q, box, rc, alpha, kmax, want_force=True, want_energy=True):
        """sqeq_coulomb_ewald: regular Ewald, reciprocal part summed over |m_d| <= kmax[d]."""
        n = pos.shape[0]
        phi = torch.empty(n, dtype=torch.float32, device=self.device)
        force = torch.empty((n, 3), dtype=torch.float32, device=self.device) if want_force else None
        e = ctypes.c_double()
        self._check(load().sqeq_coulomb_ewald(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                              _ptr(q, torch.float32, n), _box(box), float(rc), float(alpha), _grid(kmax),
                                              _ptr(phi, torch.float32, n), _ptr(force, torch.float32, 3 * n) if want_force else None,
                                              ctypes.byref(e) if want_energy else None))
        return phi, force, (e.value if want_energy else None)

    def coulomb_enqueue(self, nl, pos, q, box, rc, alpha, grid, order, phi, force, want_energy=True):
        """sqeq_coulomb_enqueue: no synchronisation; read the energy later with energy_fetch()."""
        n = pos.shape[0]
        self._check(load().sqeq_coulomb_enqueue(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                                _ptr(q, torch.float32, n), _box(box), float(rc), float(alpha),
                                                _grid(grid), int(order), _ptr(phi, torch.float32, n),
                                                _ptr(force, torch.float32, 3 * n) if force is not None else None,
                                                int(want_energy)))

    def geometry_set(self, nl, pos, box, rc, alpha, grid, order=6):
        """sqeq_geometry_set: prepare the positions once for many charge vectors (coulomb_fixed)."""
        n = pos.shape[0]
        self._check(load().sqeq_geometry_set(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n), _box(box),
                                             float(rc), float(alpha), _grid(grid), int(order)))

    def coulomb_fixed(self, q, phi=None, force=None, want_energy=False):
        """sqeq_coulomb_fixed: one charge vector on the geometry of geometry_set; no synchronisation."""
        n = q.shape[0]
        self._check(load().sqeq_coulomb_fixed(self.handle, n, _ptr(q, torch.float32, n),
                                              _ptr(phi, torch.float32, n) if phi is not None else None,
                                              _ptr(force, torch.float32, 3 * n) if force is not None else None,
                                              int(want_energy)))

    def coulomb_fixed_batch(self, q, phi=None):
        """sqeq_coulomb_fixed_batch: potentials of the charge vectors q[nvec][n] on the geometry of geometry_set."""
        nvec, n = q.shape
        if phi is None:
            phi = torch.empty((nvec, n), dtype=torch.float32, device=self.device)
        self._check(load().sqeq_coulomb_fixed_batch(self.handle, n, nvec, _ptr(q, torch.float32, nvec * n),
                                                    _ptr(phi, torch.float32, nvec * n)))
        return phi

    def energy_fetch(self):
        e = ctypes.c_double()
        self._check(load().sqeq_energy_fetch(self.handle, ctypes.byref(e)))
        return e.value

    def coulomb_host(self, nl, pos, q, box, rc, alpha, grid, order, phi, force, want_energy=True):
        """Same evaluation with HOST buffers (pinned CPU tensors): H2D and D2H copies inside the call."""
        n = pos.shape[0]
        for t in (pos, q, phi) + ((force,) if force is not None else ()):
            assert not t.is_cuda and t.is_contiguous() and t.dtype == torch.float32
        e = ctypes.c_double()
        self._check(load().sqeq_coulomb_host(self.handle, nl.handle, n, ctypes.c_void_p(pos.data_ptr()),
                                             ctypes.c_void_p(q.data_ptr()), _box(box), float(rc), float(alpha),
                                             _grid(grid), int(order), ctypes.c_void_p(phi.data_ptr()),
                                             ctypes.c_void_p(force.data_ptr()) if force is not None else None,
                                             ctypes.byref(e) if want_energy else None))
        return e.value if want_energy else None

    def coulomb_host_submit(self, slot, nl, pos, q, box, rc, alpha, grid, order, phi, force, want_energy=True):
        """Pipelined form of coulomb_host (slot 0 or 1): returns at once; coulomb_host_wait(slot) delivers."""
        n = pos.shape[0]
        for t in (pos, q, phi) + ((force,) if force is not None else ()):
            assert not t.is_cuda and t.is_contiguous() and t.dtype == torch.float32 and t.is_pinned()
        self._check(load().sqeq_coulomb_host_submit(self.handle, int(slot), nl.handle, n,
                                                    ctypes.c_void_p(pos.data_ptr()), ctypes.c_void_p(q.data_ptr()),
                                                    _box(box), float(rc), float(alpha), _grid(grid), int(order),
                                                    ctypes.c_void_p(phi.data_ptr()),
                                                    ctypes.c_void_p(force.data_ptr()) if force is not None else None,
                                                    1 if want_energy else 0))

    def coulomb_host_wait(self, slot, want_energy=True):
        e = ctypes.c_double()
        self._check(load().sqeq_coulomb_host_wait(self.handle, int(slot), ctypes.byref(e) if want_energy else None))
        return e.value if want_energy else None

    def coulomb_parts(self, nl, want_force=True):
        n = nl.n
        mk = lambda *s: torch.empty(s, dtype=torch.float32, device=self.device)
        pr, prc = mk(n), mk(n)
        fr, frc = (mk(n, 3), mk(n, 3)) if want_force else (None, None)
        e = ctypes.c_double()
        self._check(load().sqeq_coulomb_parts(self.handle, nl.handle, n, _ptr(pr, torch.float32),
                                              _ptr(fr, torch.float32), _ptr(prc, torch.float32),
                                              _ptr(frc, torch.float32), ctypes.byref(e)))
        return dict(phi_real=pr, F_real=fr, phi_rec=prc, F_rec=frc, E_rec=e.value)

    def pme_grid(self, which, grid):
        g = _grid(grid)
        out = torch.empty(tuple(g), dtype=torch.float32, device=self.device)
        rc = load().sqeq_pme_grid(self.handle, int(which), ctypes.c_void_p(out.data_ptr()))
        return out if rc == OK else None

    # ---- qeq_solve(chi, J, total_charge)
    def qeq_solve(self, nl, pos, box, rc, alpha, grid, order, ke, chi, J, total_charge, tol=1e-6,
                  max_iter=100, restart=0, raise_on_notconv=False):
        n = pos.shape[0]
        q = torch.empty(n, dtype=torch.float32, device=self.device)
        lam, rel = ctypes.c_double(), ctypes.c_double()
        it = ctypes.c_int()
        r = self._check(load().sqeq_qeq_solve(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                              _box(box), float(rc), float(alpha), _grid(grid), int(order),
                                              float(ke), _ptr(chi, torch.float32, n), _ptr(J, torch.float32, n),
                                              float(total_charge), float(tol), int(max_iter), int(restart),
                                              _ptr(q, torch.float32, n), ctypes.byref(lam), ctypes.byref(it),
                                              ctypes.byref(rel)),
                        allow=() if raise_on_notconv else (ENOTCONV,))
        return q, lam.value, it.value, rel.value, r == OK

    def qeq_solve_pc(self, nl, pos, box, rc, alpha, grid, order, ke, chi, J, total_charge, tol=1e-6,
                     max_iter=100, restart=0, jacobi=True, q0=None, lambda0=0.0):
        """sqeq_qeq_solve_pc: right Jacobi preconditioner and/or an initial guess (q0, lambda0)."""
        n = pos.shape[0]
        q = torch.empty(n, dtype=torch.float32, device=self.device)
        lam, rel = ctypes.c_double(), ctypes.c_double()
        it = ctypes.c_int()
        r = self._check(load().sqeq_qeq_solve_pc(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                                 _box(box), float(rc), float(alpha), _grid(grid), int(order),
                                                 float(ke), _ptr(chi, torch.float32, n), _ptr(J, torch.float32, n),
                                                 float(total_charge), float(tol), int(max_iter), int(restart),
                                                 int(bool(jacobi)), _ptr(q0, torch.float32, n) if q0 is not None else None,
                                                 float(lambda0), _ptr(q, torch.float32, n), ctypes.byref(lam),
                                                 ctypes.byref(it), ctypes.byref(rel)), allow=(ENOTCONV,))
        return q, lam.value, it.value, rel.value, r == OK

    # ---- regular Born-Oppenheimer MD
    def bomd_init(self, nl, pos, box, params, chi, u, tol=1e-6, max_iter=100, jacobi=True):
        """Returns the state (q fp64 [n], lambda), the force and [U_BO, 0, relres, evaluations]."""
        n = pos.shape[0]
        q = torch.zeros(n, dtype=torch.float64, device=self.device)
        force = torch.empty((n, 3), dtype=torch.float32, device=self.device)
        lam = ctypes.c_double(0.0)
        en = (ctypes.c_double * 4)()
        r = self._check(load().sqeq_bomd_init(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n), _box(box),
                                              ctypes.byref(params), _ptr(chi, torch.float32, n), _ptr(u, torch.float32, n),
                                              float(tol), int(max_iter), int(bool(jacobi)), ctypes.c_void_p(q.data_ptr()),
                                              ctypes.byref(lam), _ptr(force, torch.float32), en), allow=(ENOTCONV,))
        return dict(q=q, lam=lam, converged=r == OK), force, list(en)

    def bomd_step(self, nl, pos, vel, mass, box, params, chi, u, state, force, tol=1e-6, max_iter=100, jacobi=True,
                  warm_start=True):
        n = pos.shape[0]
        en = (ctypes.c_double * 4)()
        r = self._check(load().sqeq_bomd_step(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                              _ptr(vel, torch.float32, 3 * n), _ptr(mass, torch.float32, n), _box(box),
                                              ctypes.byref(params), _ptr(chi, torch.float32, n), _ptr(u, torch.float32, n),
                                              float(tol), int(max_iter), int(bool(jacobi)), int(bool(warm_start)),
                                              ctypes.c_void_p(state["q"].data_ptr()), ctypes.byref(state["lam"]),
                                              _ptr(force, torch.float32, 3 * n), en), allow=(ENOTCONV,))
        state["converged"] = r == OK
        return list(en)

    # ---- shadow XL-BOMD
    def shadow_md_init(self, nl, pos, box, params, chi, u, tol=1e-8, max_iter=200, n0=None):
        """n0 given (numpy/torch fp64 [n]) with max_iter=0: start the history from n0 instead of q_min."""
        n = pos.shape[0]
        nhist = torch.zeros((7, n), dtype=torch.float64, device=self.device)
        if n0 is not None:
            nhist[0] = torch.as_tensor(n0, dtype=torch.float64).to(self.device)
        force = torch.empty((n, 3), dtype=torch.float32, device=self.device)
        en = (ctypes.c_double * 4)()
        self._check(load().sqeq_shadow_md_init(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                               _box(box), ctypes.byref(params), _ptr(chi, torch.float32, n),
                                               _ptr(u, torch.float32, n), float(tol), int(max_iter),
                                               ctypes.c_void_p(nhist.data_ptr()), _ptr(force, torch.float32),
                                               en))
        return nhist, force, list(en)

    def shadow_md_step(self, nl, pos, vel, mass, box, params, chi, u, nhist, force, want_energies=True):
        n = pos.shape[0]
        en = (ctypes.c_double * 4)()
        self._check(load().sqeq_shadow_md_step(self.handle, nl.handle, n, _ptr(pos, torch.float32, 3 * n),
                                               _ptr(vel, torch.float32, 3 * n), _ptr(mass, torch.float32, n),
                                               _box(box), ctypes.byref(params), _ptr(chi, torch.float32, n),
                                               _ptr(u, torch.float32, n), ctypes.c_void_p(nhist.data_ptr()),
                                               _ptr(force, torch.float32, 3 * n),
                                               en if want_energies else None))
        return list(en) if want_energies else None

    def shadow_md_run(self, nl, pos, vel, mass, box, params, chi, u, nhist, force, nsteps, slack=0.05):
        """sqeq_shadow_md_run: nsteps steps, the list rebuilt by the library when the drift would reach skin/2 - slack.
        `nl` is updated in place (its handle may be replaced).  Returns the stats dict."""
        n = pos.shape[0]
        st = (ctypes.c_double * 8)()
        h = ctypes.c_void_p(nl.handle.value)
        try:
            self._check(load().sqeq_shadow_md_run(self.handle, ctypes.byref(h), n, _ptr(pos, torch.float32, 3 * n),
                                                  _ptr(vel, torch.float32, 3 * n), _ptr(mass, torch.float32, n), _box(box),
                                                  ctypes.byref(params), _ptr(chi, torch.float32, n), _ptr(u, torch.float32, n),
                                                  ctypes.c_void_p(nhist.data_ptr()), _ptr(force, torch.float32, 3 * n),
                                                  int(nsteps), float(nl.cutoff), float(slack), st))
        finally:
            nl.handle = h
        keys = ["U", "ekin", "resnorm", "evals_last_step", "rebuilds", "max_ahead_accepted", "drift_end", "half_skin"]
        return dict(zip(keys, list(st)))

    # ---- timing
    def profile_enable(self, on=True):
        self._check(load().sqeq_profile_enable(self.handle, int(on)))

    def profile_reset(self):
        self._check(load().sqeq_profile_reset(self.handle))

    def profile_read(self):
        out = {}
        for k, name in enumerate(STAGES):
            ms, cnt = ctypes.c_double(), ctypes.c_int64()
            self._check(load().sqeq_profile_read(self.handle, k, ctypes.byref(ms), ctypes.byref(cnt)))
            out[name] = (ms.value, cnt.value)
        return out

    def set_option(self, name, value):
        self._check(load().sqeq_set_option(self.handle, name.encode(), int(value)))

    def launch_count(self, reset=False):
        c = ctypes.c_int64()
        self._check(load().sqeq_launch_count(self.handle, ctypes.byref(c), int(reset)))
        return c.value


NOALLOC_MAX_N = 4194304


def energy_noalloc(q, phi, out, stream=None):
    """sqeq_energy_noalloc: out (device float64 tensor of one element) <- 1/2 sum q phi on `stream`; allocates nothing."""
    dev = q.device
    if stream is None:
        stream = torch.cuda.current_stream(dev)
    n = q.shape[0]
    if out.dtype != torch.float64 or out.numel() != 1 or not out.is_cuda:
        raise ValueError("out must be a CUDA float64 tensor with one element")
    rc_ = load().sqeq_energy_noalloc(dev.index or 0, ctypes.c_void_p(stream.cuda_stream), n, _ptr(q, torch.float32, n),
                                     _ptr(phi, torch.float32, n), ctypes.c_void_p(out.data_ptr()))
    if rc_ != OK:
        raise SqeqError(rc_, load().sqeq_last_error(None).decode())
    return out


def ewald_params(box, rc, delta):
    """sqeq_ewald_params: (alpha, kmax[3], grid[3]) for an Ewald accuracy delta (OpenMM's heuristics)."""
    a = ctypes.c_double()
    km, gr = (ctypes.c_int * 3)(), (ctypes.c_int * 3)()
    rc_ = load().sqeq_ewald_params(_box(box), float(rc), float(delta), ctypes.byref(a), km, gr)
    if rc_ != OK:
        raise SqeqError(rc_, "sqeq_ewald_params: bad argument")
    return a.value, list(km), list(gr)


def md_params(cfg, dt=0.5, ke=14.3996454784255, total_charge=0.0, krylov_rank=4,
              k_oh=48.0, r_oh=0.9572, k_hh=10.0, r_hh=1.5139, krylov_tol=0.0, k_rep=0.0, r_rep=0.0):
    """sqeq_md_params for a workloads.Config with the XL-BOMD constants of DESIGN.md R-MD."""
    p = MdParams()
    p.dt, p.ke, p.total_charge = dt, ke, total_charge
    p.rc, p.alpha = cfg.rc, cfg.alpha
    p.grid[:] = [cfg.grid] * 3
    p.order, p.krylov_rank = cfg.order, krylov_rank
    p.k_oh, p.r_oh, p.k_hh, p.r_hh = k_oh, r_oh, k_hh, r_hh
    p.kappa, p.alpha_diss = 1.82, 0.018
    p.c[:] = [-6.0, 14.0, -8.0, -3.0, 4.0, -1.0, 0.0]
    p.krylov_tol, p.k_rep, p.r_rep = krylov_tol, k_rep, r_rep
    return p
